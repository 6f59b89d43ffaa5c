"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module is the ONE thing the CUDA path's tests/bench and the CPU oracle's tests share: it only
*generates inputs* (grid / crystal / beam parameter dictionaries, the fp32 temperature array, the
complex64 input envelope).  It contains none of the method's arithmetic (no transform, no propagator,
no coupled-wave step) and imports neither the CUDA binding nor the oracle.

The paper's workload: cw 1064 nm -> 532 nm, focused TEM00 pump, w_F = 29 um,
xi = 2.84, ~30 mm MgO:sPPLT crystal, oven at 56.5 C, pump up to 30 W.  No public dataset is involved;
every array is produced here from ``numpy.random.default_rng(seed)`` (PCG64) and handed identically to
both paths: ``T`` as float32, ``A1`` rounded to complex64 before either path reads it.
"""
from __future__ import annotations

import math

import numpy as np

EPS0 = 8.8541878128e-12
C0 = 299792458.0
T_PM = 56.5   # oven temperature quoted at PAPER.md:292; only T - T_pm enters the model

CONFIG_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")
STREAM_NAMES = ("stream256", "stream1024")   # working set larger than L2


def crystal(L, alpha=False, ddk_dT=0.0, **over):
    c = dict(L=L, lambda1=1064e-9, n1=2.14, n2=2.18, d_eff=10e-12, dk0=0.0, ddk_dT=ddk_dT, T_pm=T_PM,
             alpha1=0.0, alpha2=0.0, beta1=0.0, beta2=0.0)
    if alpha:   # "absorption as in config 2"
        c.update(alpha1=0.1, alpha2=1.0, beta1=0.0, beta2=1e-11)
    c.update(over)
    return c


def k1_of(c):
    return 2.0 * math.pi * c["n1"] / c["lambda1"]


def waist_for_xi(c, xi):
    """xi = L / (2 zR), zR = k1 w0^2 / 2  ->  w0 = sqrt(L / (xi k1))."""
    return math.sqrt(c["L"] / (xi * k1_of(c)))


def beam(c, P, xi, window_w0, focus_z=None):
    w0 = waist_for_xi(c, xi)
    return dict(P=P, w0=w0, focus_z=c["L"] / 2 if focus_z is None else focus_z,
                lx=window_w0 * w0, ly=window_w0 * w0)


def axes(nx, ny, bm):
    dx, dy = bm["lx"] / nx, bm["ly"] / ny
    x = (np.arange(nx) - nx // 2) * dx
    y = (np.arange(ny) - ny // 2) * dy
    return x, y


def gaussian_pump(nx, ny, c, bm):
    """Input envelope of PAPER.md:104 (Eq. 6), any focus via Eq. 5; complex64 [ny][nx].

    |A_F0|^2 = 4 P / (eps0 c n1 pi w0^2) so that the analytic beam carries P (I = eps0 c n |A|^2 / 2,
    PAPER.md:120).  No renormalisation of the clipped discrete sum.
    """
    x, y = axes(nx, ny, bm)
    zR = 0.5 * bm["w0"] ** 2 * k1_of(c)
    q = 1.0 + 1j * (-bm["focus_z"] / zR)
    A0 = math.sqrt(4.0 * bm["P"] / (EPS0 * C0 * c["n1"] * math.pi * bm["w0"] ** 2))
    r2 = x[None, :] ** 2 + y[:, None] ** 2
    return ((A0 / q) * np.exp(-r2 / (bm["w0"] ** 2 * q))).astype(np.complex64)


def noisy_sh_seed(nx, ny, rms_amplitude, seed, batch=1):
    """Second-harmonic input of PAPER.md:106 ("A_SH(z=0) ... Gaussian white noise with both random amplitude and
    phase"; setNoisyField): independent circular complex Gaussian samples, E|A|^2 =
    rms_amplitude^2 at every grid point.  The paper gives no level, so the amplitude is an explicit argument (V/m);
    the BASELINE configs use A_SH(0) = 0 instead.  complex64 [batch][ny][nx], numpy PCG64 from `seed`."""
    rng = np.random.default_rng(seed)
    z = rng.standard_normal((batch, ny, nx, 2))
    return ((rms_amplitude / math.sqrt(2.0)) * (z[..., 0] + 1j * z[..., 1])).astype(np.complex64)


def _bump_field(nx, ny, nzt, c, bm, seed, grad_K=1.0, nbump=8):
    """T_pm + sum of `nbump` isotropic 3-D Gaussian bumps (amplitude U(0,3) K, 1/e radius U(0.5,2) mm,
    centres uniform over window x [0,L]) + grad_K * z/L.  float32 [nzt][ny][nx]."""
    rng = np.random.default_rng(seed)
    amp = rng.uniform(0.0, 3.0, nbump)
    wid = rng.uniform(0.5e-3, 2.0e-3, nbump)
    cx = rng.uniform(-bm["lx"] / 2, bm["lx"] / 2, nbump)
    cy = rng.uniform(-bm["ly"] / 2, bm["ly"] / 2, nbump)
    cz = rng.uniform(0.0, c["L"], nbump)
    x, y = axes(nx, ny, bm)
    z = np.linspace(0.0, c["L"], nzt)
    T = np.empty((nzt, ny, nx), dtype=np.float32)
    ex = [np.exp(-((x - cx[b]) / wid[b]) ** 2) for b in range(nbump)]
    ey = [np.exp(-((y - cy[b]) / wid[b]) ** 2) for b in range(nbump)]
    ez = [amp[b] * np.exp(-((z - cz[b]) / wid[b]) ** 2) for b in range(nbump)]
    # plane by plane keeps the fp64 temporary at one plane (cfg5: 1 GiB of fp32 output)
    for k in range(nzt):
        plane = np.full((ny, nx), T_PM + grad_K * z[k] / c["L"])
        for b in range(nbump):
            plane += ez[b][k] * (ey[b][:, None] * ex[b][None, :])
        T[k] = plane
    return T


def make(name: str, nz: int | None = None, batch: int | None = None):
    """Return one workload: dict(name, grid, crystal, beams, T, T_uniform, per_member, A1).

    ``nz`` overrides the step count (reduced-length parity cases); the temperature planes are then
    regenerated on the new nodes for the configs whose planes sit on the nodes (cfg2, cfg3).
    ``batch`` overrides the member count of cfg4 (first `batch` members of the 8x8 sweep).
    """
    name = name.lower()
    T = None
    T_uniform = T_PM
    per_member = False
    if name == "cfg1":
        nx = ny = 64
        nzs = 200 if nz is None else nz
        c = crystal(30e-3)
        beams = [beam(c, 5.0, 2.84, 6.0)]
        nzt = 0
    elif name == "cfg2":
        nx = ny = 128
        nzs = 1000 if nz is None else nz
        c = crystal(30e-3, alpha=True, ddk_dT=-30.0)
        bm = beam(c, 30.0, 2.84, 6.0)
        beams = [bm]
        nzt = nzs + 1
        rng = np.random.default_rng(2)
        x, y = axes(nx, ny, bm)
        r2 = x[None, :] ** 2 + y[:, None] ** 2
        zR = 0.5 * bm["w0"] ** 2 * k1_of(c)
        T = np.empty((nzt, ny, nx), dtype=np.float32)
        for k in range(nzt):
            z = c["L"] * k / (nzt - 1)
            wz = bm["w0"] * math.sqrt(1.0 + ((z - c["L"] / 2) / zR) ** 2)
            T[k] = (T_PM + 2.0 * np.exp(-2.0 * r2 / (3.0 * wz) ** 2) * (0.5 + 0.5 * z / c["L"])
                    + rng.uniform(-0.01, 0.01, (ny, nx)))
    elif name == "cfg3":
        nx = ny = 256
        nzs = 4000 if nz is None else nz
        c = crystal(50e-3, alpha=True, ddk_dT=-30.0)
        bm = beam(c, 50.0, 1.0, 8.0)
        beams = [bm]
        nzt = nzs + 1
        T = _bump_field(nx, ny, nzt, c, bm, seed=3)
    elif name == "cfg4":
        nx = ny = 128
        nzs = 1000 if nz is None else nz
        c = crystal(30e-3, alpha=True, ddk_dT=-30.0)
        xis = np.geomspace(0.2, 10.0, 8)
        Ps = np.geomspace(1.0, 100.0, 8)
        beams = [beam(c, float(Ps[ip]), float(xis[ix]), 6.0) for ix in range(8) for ip in range(8)]
        if batch is not None:
            beams = beams[:batch]
        nzt = 0
        T_uniform = T_PM + 0.5
    elif name == "cfg5":
        nx = ny = 1024
        nzs = 10000 if nz is None else nz
        c = crystal(40e-3, alpha=True, ddk_dT=-30.0)
        bm = beam(c, 100.0, 2.84, 10.0)
        beams = [bm]
        nzt = 256
        T = _bump_field(nx, ny, nzt, c, bm, seed=5)
    elif name in ("stream256", "stream1024"):
        # Throughput regime: a sweep whose field state (16 B/pt) is larger than the
        # 126 MB L2, so every pass really streams through HBM.  Members: pump power log-spaced over 1-100 W at
        # xi = 2.84 in the cfg2 / cfg5 crystal, uniform T_pm + 0.5 K (as cfg4), each on its own window.
        nx = ny = 256 if name == "stream256" else 1024
        members = (192 if nx == 256 else 16) if batch is None else batch       # 201 MB / 268 MB of fields
        nzs = 200 if nz is None else nz
        c = crystal(30e-3 if nx == 256 else 40e-3, alpha=True, ddk_dT=-30.0)
        beams = [beam(c, float(P), 2.84, 8.0 if nx == 256 else 10.0) for P in np.geomspace(1.0, 100.0, members)]
        nzt = 0
        T_uniform = T_PM + 0.5
    else:
        raise ValueError("unknown workload %r" % name)
    grid = dict(nx=nx, ny=ny, nz=nzs, nzt=nzt, batch=len(beams))
    A1 = np.stack([gaussian_pump(nx, ny, c, b) for b in beams])
    return dict(name=name, grid=grid, crystal=c, beams=beams, T=T, T_uniform=T_uniform,
                per_member=per_member, A1=A1)


def algorithmic_bytes_per_point_step(w) -> float:
    """Bytes the METHOD must move per grid-point z-step if the state does not live on chip
    (SURVEY.md §8(d)): read+write A1, A2 (32 B); with a temperature array also phi read+write (8 B)
    and the share of the T planes (4 B x planes consumed per step)."""
    g = w["grid"]
    b = 32.0
    if g["nzt"] >= 1:
        b += 8.0 + 4.0 * (g["nzt"] if g["nzt"] > 1 else 1) / g["nz"]
    return b


def algorithmic_flops_per_point_step(w) -> float:
    """40 log2(N) + 330: four 2-D FFTs at 10 log2 N (radix-2 count) + phase
    multiplies + RK4 + 3 sincos + T/dk/phi + power."""
    g = w["grid"]
    return 20.0 * (math.log2(g["nx"]) + math.log2(g["ny"])) + 330.0
