"""Pins of the CPU oracle against what the paper and the mathematics fix (never against itself).

Each test names the passage of /root/reference/PAPER.md ("P:n") or the closed form it checks, and is
chosen so that a plausible slip in the oracle (dropped term, wrong sign/index, transposed operand, the
printed-but-inconsistent kappa_SH) fails at least one of them.  CPU only.
"""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_2410_04994_b200 import workloads as wl

EPS0, C0 = 8.8541878128e-12, 299792458.0


def rel_l2(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


# ------------------------------------------------------------------------------------------------
# 1. transforms: definition, library routine, closed forms
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ny,nx", [(2, 2), (4, 4), (4, 8), (8, 4), (16, 16), (2, 16), (16, 8)])
def test_fft_matches_brute_force_dft_and_numpy(ny, nx):
    rng = np.random.default_rng(100 + ny * 31 + nx)
    a = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    for sign, ref in ((-1, np.fft.fft2(a)), (+1, np.fft.ifft2(a))):
        fast = oracle.fft2(a, sign)
        brute = oracle.dft2_brute(a, sign)
        assert rel_l2(fast, brute) < 1e-12          # own FFT == the written-out definition
        assert rel_l2(brute, ref) < 1e-12           # the definition == the library routine (sign, 1/N)
    assert rel_l2(oracle.fft2(oracle.fft2(a, -1), +1), a) < 1e-12
    # Parseval for the unnormalised forward transform
    assert abs(np.sum(np.abs(oracle.fft2(a, -1)) ** 2) / (nx * ny) / np.sum(np.abs(a) ** 2) - 1) < 1e-12


def test_fft_closed_forms_fix_sign_and_axis_order():
    ny, nx = 8, 16
    # a plane wave e^{+2 pi i (3 x/nx + 5 y/ny)} goes to the single bin [ky=5][kx=3] with weight nx*ny
    y, x = np.mgrid[0:ny, 0:nx]
    a = np.exp(2j * np.pi * (3 * x / nx + 5 * y / ny))
    F = oracle.fft2(a, -1)
    expect = np.zeros((ny, nx), complex)
    expect[5, 3] = nx * ny
    assert np.max(np.abs(F - expect)) < 1e-10
    # a delta at (y0, x0) goes to e^{-2 pi i (kx x0/nx + ky y0/ny)}
    d = np.zeros((ny, nx), complex)
    d[2, 7] = 1.0
    ky, kx = np.mgrid[0:ny, 0:nx]
    assert np.max(np.abs(oracle.fft2(d, -1) - np.exp(-2j * np.pi * (kx * 7 / nx + ky * 2 / ny)))) < 1e-12


# ------------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------------
def plane_wave_case(A0, nz, L=30e-3, n=4, **cr):
    c = wl.crystal(L, **cr)
    bm = dict(P=0.0, w0=1.0, focus_z=0.0, lx=1e-3, ly=1e-3)
    g = dict(nx=n, ny=n, nz=nz, nzt=0)
    A1 = np.full((1, n, n), A0, dtype=np.complex128)
    return g, c, bm, A1


# ------------------------------------------------------------------------------------------------
# 2. linear step: free diffraction of Eq. 6 must reproduce Eq. 5, w(z) and the Gouy phase
# ------------------------------------------------------------------------------------------------
def eq5_envelope(x, y, z, c, bm):
    """Eq. 5 without the carrier e^{i k z}, retyped here from the paper (not from the oracle)."""
    k1 = 2 * np.pi * c["n1"] / c["lambda1"]
    zR = bm["w0"] ** 2 * k1 / 2
    tau = (z - bm["focus_z"]) / zR
    A0 = math.sqrt(4 * bm["P"] / (EPS0 * C0 * c["n1"] * np.pi * bm["w0"] ** 2))
    r2 = x[None, :] ** 2 + y[:, None] ** 2
    return A0 / (1 + 1j * tau) * np.exp(-r2 / (bm["w0"] ** 2 * (1 + 1j * tau)))


def test_free_diffraction_matches_analytic_gaussian_beam():
    c = wl.crystal(30e-3, d_eff=0.0)
    bm = wl.beam(c, 5.0, 2.84, 40.0)
    n = 256
    x, y = wl.axes(n, n, bm)
    A_in = oracle.gaussian_input(dict(nx=n, ny=n, nz=1, nzt=0), c, bm)
    # the oracle's Eq. 6 generator against the formula typed from the paper (xi form)
    k1 = 2 * np.pi * c["n1"] / c["lambda1"]
    xi = c["L"] / (bm["w0"] ** 2 * k1)
    A0 = math.sqrt(4 * bm["P"] / (EPS0 * C0 * c["n1"] * np.pi * bm["w0"] ** 2))
    eq6 = A0 / (1 - 1j * xi) * np.exp(-(x[None, :] ** 2 + y[:, None] ** 2) / (bm["w0"] ** 2 * (1 - 1j * xi)))
    assert rel_l2(A_in, eq6) < 1e-13
    assert abs(xi - 2.84) < 1e-12
    zR = bm["w0"] ** 2 * k1 / 2
    for nz, frac in ((8, 0.5), (16, 1.0)):      # stop at the focus and at the exit face
        cc = dict(c, L=c["L"] * frac)
        # keep the focus where it was (L/2 of the full crystal)
        o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), cc, [bm])
        A1, A2 = o.propagate(A_in[None])
        ref = eq5_envelope(x, y, cc["L"], c, bm)
        assert rel_l2(A1[0], ref) < 1e-10
        assert np.max(np.abs(A2)) == 0.0
        # beam radius from the second moment: sqrt(2 <r^2>) = w0 sqrt(1 + tau^2)
        I = np.abs(A1[0]) ** 2
        r2 = x[None, :] ** 2 + y[:, None] ** 2
        w_meas = math.sqrt(2 * np.sum(I * r2) / np.sum(I))
        tau = (cc["L"] - bm["focus_z"]) / zR
        assert abs(w_meas / (bm["w0"] * math.sqrt(1 + tau ** 2)) - 1) < 1e-9
        # on-axis (Gouy) phase relative to the input: -(atan tau - atan tau0)
        tau0 = -bm["focus_z"] / zR
        dphi = np.angle(A1[0][n // 2, n // 2] / A_in[n // 2, n // 2])
        expect = -(math.atan(tau) - math.atan(tau0))
        assert abs((dphi - expect + np.pi) % (2 * np.pi) - np.pi) < 1e-9
    # survey's scratch value of the Gouy phase at the exit face (SURVEY.md §8(c) pin table): -2.46448
    assert abs(expect - (-2.46448)) < 1e-5


def test_sh_field_diffracts_with_its_own_wavevector():
    """k2 = 2 pi n2 / (lambda1/2): a SH Gaussian must follow Eq. 5 with k2, not k1."""
    c = wl.crystal(20e-3, d_eff=0.0)
    n = 128
    w0 = 25e-6
    bm = dict(P=1.0, w0=w0, focus_z=0.0, lx=30 * w0, ly=30 * w0)
    x, y = wl.axes(n, n, bm)
    r2 = x[None, :] ** 2 + y[:, None] ** 2
    A2_in = np.exp(-r2 / w0 ** 2).astype(complex)
    o = oracle.Oracle(dict(nx=n, ny=n, nz=4, nzt=0), c, [bm])
    A1, A2 = o.propagate(np.zeros((1, n, n), complex), A2_in[None])
    k2 = 2 * np.pi * c["n2"] / (c["lambda1"] / 2)
    tau = c["L"] / (w0 ** 2 * k2 / 2)
    ref = 1 / (1 + 1j * tau) * np.exp(-r2 / (w0 ** 2 * (1 + 1j * tau)))
    assert rel_l2(A2[0], ref) < 1e-10
    assert np.max(np.abs(A1)) == 0.0


# ------------------------------------------------------------------------------------------------
# 3. absorption: P_j(z) = P_j(0) exp(-alpha_j z)   (L_j of P:143 with d_eff = beta = 0)
# ------------------------------------------------------------------------------------------------
def test_linear_absorption_is_exact():
    c = wl.crystal(30e-3, d_eff=0.0, alpha1=3.0, alpha2=11.0)
    bm = wl.beam(c, 2.0, 1.5, 12.0)
    n, nz = 32, 10
    A_in = wl.gaussian_pump(n, n, c, bm).astype(np.complex128)
    o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), c, [bm])
    o.propagate(A_in[None], 0.5j * A_in[None])
    h = o.power_history()
    z = np.linspace(0, c["L"], nz + 1)
    assert np.max(np.abs(h[:, 0] / h[0, 0] / np.exp(-3.0 * z) - 1)) < 1e-12
    assert np.max(np.abs(h[:, 1] / h[0, 1] / np.exp(-11.0 * z) - 1)) < 1e-12
    p1, p2 = o.power(0, c["L"])
    assert p1 == h[-1, 0] and p2 == h[-1, 1]


# ------------------------------------------------------------------------------------------------
# 4. coupling constants + RK4: energy conservation (kills the printed kappa_SH, G2)
# ------------------------------------------------------------------------------------------------
def test_total_power_conserved_without_absorption():
    w = wl.make("cfg1")
    o = oracle.Oracle(w["grid"], w["crystal"], w["beams"])
    o.propagate(w["A1"].astype(np.complex128))
    h = o.power_history()
    tot = h.sum(axis=1)
    assert np.max(np.abs(tot / tot[0] - 1)) < 1e-9          # north_star pin 3
    assert h[-1, 1] / tot[0] > 0.05                         # and there is real conversion going on
    # indicative values of an independent fp64 implementation (numpy-FFT scratch run)
    assert abs(h[0, 0] - 4.54715) < 2e-5
    assert abs(h[-1, 1] / tot[0] - 0.0737969) < 2e-6
    assert abs(h[-1, 0] / h[0, 0] - 0.926203) < 2e-6


# ------------------------------------------------------------------------------------------------
# 5. plane-wave depletion: P2/P0 = tanh^2(Gamma L)
# ------------------------------------------------------------------------------------------------
def test_plane_wave_depletion_tanh2():
    A0 = 3e6
    g, c, bm, A1 = plane_wave_case(A0, nz=400)
    o = oracle.Oracle(g, c, [bm])
    o.propagate(A1)
    h = o.power_history()
    I0 = EPS0 * C0 * c["n1"] * A0 ** 2 / 2
    Gamma = math.sqrt(8 * np.pi ** 2 * c["d_eff"] ** 2 * I0 /
                      (EPS0 * C0 * c["n1"] ** 2 * c["n2"] * c["lambda1"] ** 2))
    expect = math.tanh(Gamma * c["L"]) ** 2
    assert abs(h[-1, 1] / h[0, 0] - expect) < 1e-9
    assert abs(expect - 0.97126055858) < 1e-9               # SURVEY.md §8(c) scratch value
    # along z as well
    z = np.linspace(0, c["L"], g["nz"] + 1)
    assert np.max(np.abs(h[:, 1] / h[0, 0] - np.tanh(Gamma * z) ** 2)) < 1e-9


# ------------------------------------------------------------------------------------------------
# 6. mismatch phase: sinc^2, every encoding of the same uniform temperature, linear-in-z temperature
# ------------------------------------------------------------------------------------------------
def sinc2_expect(c, A0, dk):
    kappa2 = 2 * np.pi * c["d_eff"] / (c["n2"] * c["lambda1"])
    xarg = dk * c["L"] / 2
    return (c["n2"] / c["n1"]) * kappa2 ** 2 * A0 ** 2 * c["L"] ** 2 * (math.sin(xarg) / xarg) ** 2


def test_uniform_mismatch_sinc2_for_every_temperature_encoding():
    A0, nz, n = 1.0, 512, 4
    dT = 1.5                                   # 56.5 + 1.5 = 58.0 is exact in fp32
    g, c, bm, A1 = plane_wave_case(A0, nz, dk0=150.0, ddk_dT=-30.0)
    dk = 150.0 - 30.0 * dT
    expect = sinc2_expect(c, A0, dk)
    results = []
    for nzt in (0, 1, 2, 5, nz + 1):
        gg = dict(g, nzt=nzt)
        o = oracle.Oracle(gg, c, [bm])
        if nzt == 0:
            o.set_temperature(None, wl.T_PM + dT)
        else:
            o.set_temperature(np.full((nzt, n, n), wl.T_PM + dT, np.float32))
        o.propagate(A1)
        h = o.power_history()
        results.append(h[-1, 1] / h[0, 0])
    for r in results:
        assert abs(r / expect - 1) < 1e-8
    assert np.ptp(results) / expect < 1e-12
    # the guard: dk0 alone, or dk0 - g dT, would give clearly different values
    assert abs(sinc2_expect(c, A0, 150.0) / expect - 1) > 0.5
    assert abs(sinc2_expect(c, A0, 150.0 + 30.0 * dT) / expect - 1) > 0.5


def test_linear_in_z_temperature_gives_quadratic_phase():
    """T = T_pm + a z/L  ->  dk = g a z / L, phi = g a z^2 / (2L) (Eq. 3); undepleted SH power is
    (n2/n1) kappa2^2 A0^2 |int_0^L e^{i phi(z)} dz|^2, integral by independent quadrature."""
    A0, nz, n = 1.0, 512, 4
    a, gcoef = 2.0, -150.0
    g, c, bm, A1 = plane_wave_case(A0, nz, ddk_dT=gcoef, T_pm=0.0)
    L = c["L"]
    re = integrate.quad(lambda z: math.cos(gcoef * a * z * z / (2 * L)), 0, L, epsabs=1e-16, epsrel=1e-13)[0]
    im = integrate.quad(lambda z: math.sin(gcoef * a * z * z / (2 * L)), 0, L, epsabs=1e-16, epsrel=1e-13)[0]
    kappa2 = 2 * np.pi * c["d_eff"] / (c["n2"] * c["lambda1"])
    expect = (c["n2"] / c["n1"]) * kappa2 ** 2 * A0 ** 2 * (re * re + im * im)
    vals = []
    for nzt in (2, 9, nz + 1):                 # a linear profile is exact under linear interpolation
        planes = np.linspace(0.0, a, nzt)      # multiples of 2^-k: exact in fp32
        T = np.broadcast_to(planes[:, None, None], (nzt, n, n)).astype(np.float32)
        o = oracle.Oracle(dict(g, nzt=nzt), c, [bm]).set_temperature(T)
        o.propagate(A1)
        h = o.power_history()
        vals.append(h[-1, 1] / h[0, 0])
    for v in vals:
        assert abs(v / expect - 1) < 1e-8
    # a per-point different temperature must stay per-point: two columns with different slopes
    T = np.zeros((nz + 1, n, n), np.float32)
    T[:, :, 2:] = np.linspace(0.0, a, nz + 1)[:, None, None]
    # (a 10 m window switches diffraction off, so the columns do not talk to each other)
    o = oracle.Oracle(dict(g, nzt=nz + 1), c, [dict(bm, lx=10.0, ly=10.0)]).set_temperature(T)
    _, A2 = o.propagate(A1)
    p_cold = np.abs(A2[0][:, :2]) ** 2          # |A2(L)|^2 = kappa2^2 A0^4 |int e^{i phi}|^2
    p_hot = np.abs(A2[0][:, 2:]) ** 2
    assert np.max(np.abs(p_hot / (kappa2 ** 2 * A0 ** 4 * (re * re + im * im)) - 1)) < 1e-8
    assert np.max(np.abs(p_cold / (kappa2 ** 2 * A0 ** 4 * L * L) - 1)) < 1e-8


def exact_phase_integral(dk_planes, L):
    """int_0^L e^{i phi(z)} dz for a mismatch that is piecewise LINEAR in z between equidistant planes (T is linearly
    interpolated between its planes, G15), phi(z) = int_0^z dk (Eq. 3) hence piecewise quadratic.  Independent
    of the oracle: adaptive quadrature (scipy) interval by interval on the closed-form phase."""
    nzt = len(dk_planes)
    hk = L / (nzt - 1)
    phi0 = 0.0
    tot = 0.0 + 0.0j
    for k in range(nzt - 1):
        a, b = float(dk_planes[k]), float(dk_planes[k + 1])
        ph = lambda s, a=a, b=b, phi0=phi0: phi0 + a * s + (b - a) * s * s / (2 * hk)
        re = integrate.quad(lambda s: math.cos(ph(s)), 0.0, hk, epsabs=0.0, epsrel=1e-13)[0]
        im = integrate.quad(lambda s: math.sin(ph(s)), 0.0, hk, epsabs=0.0, epsrel=1e-13)[0]
        tot += re + 1j * im
        phi0 += 0.5 * (a + b) * hk
    return tot


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("profile", ["linear", "planes"])
def test_complex_sh_amplitude_pins_the_phase_samples_inside_a_step(scheme, profile):
    """Undepleted plane wave, no absorption: A1 stays A0 and Eq. 2 reduces to the quadrature
        A2(L) = i kappa2 A0^2 int_0^L e^{i phi(z)} dz,   phi = int_0^z dk dz'   (Eq. 3).
    An RK4 step on a pure quadrature is Simpson's rule, so with the phase sampled where G15 puts it (z_n,
    z_n + dz/2, z_n + dz of the in-step quadratic; scheme 1: the two half-steps of Eq. 14-15, sample at
    0, dz/4, dz/2 and dz/2, 3dz/4, dz) the error is O(dz^4); a sample taken anywhere else is O(dz^2) or worse, and a
    phase that does not accumulate from step to step is an O(1) error.  The COMPLEX amplitude is compared: |A2|^2
    alone hides a mid-step phase error at first order."""
    A0, n, nz = 3.0e3, 4, 512
    gcoef = -40.0
    g, c, bm, A1 = plane_wave_case(A0, nz, dk0=25.0, ddk_dT=gcoef, T_pm=0.0)
    L = c["L"]
    if profile == "linear":
        nzt = 2
        planes = np.array([0.5, 2.5])                        # T linear in z: dk from 5 to -75 rad/m
    else:
        nzt = 9                                              # 8 plane intervals, 64 steps each: a profile that is
        planes = np.array([0.0, 1.75, 0.5, 2.25, 2.0, -0.75, 0.25, 1.5, 3.0])   # not linear (nor monotone) in z
    T = np.broadcast_to(planes[:, None, None], (nzt, n, n)).astype(np.float32)   # multiples of 1/4: exact in fp32
    expect = 1j * (2 * np.pi * c["d_eff"] / (c["n2"] * c["lambda1"])) * A0 ** 2 * \
        exact_phase_integral(25.0 + gcoef * planes, L)
    res = {}
    for steps in (nz // 2, nz):
        o = oracle.Oracle(dict(g, nz=steps, nzt=nzt), c, [bm], scheme=scheme, undepleted=True).set_temperature(T)
        B1, B2 = o.propagate(A1)
        assert np.max(np.abs(B1 - A0)) == 0.0                # the pump really is untouched
        assert np.ptp(B2.real) == 0.0 and np.ptp(B2.imag) == 0.0
        res[steps] = B2[0, 0, 0]
    err = {k: abs(v / expect - 1) for k, v in res.items()}
    assert err[nz] < 1e-9, err                               # measured ~1e-11
    assert err[nz // 2] < 16 * 1.3 * max(err[nz], 1e-12) + 1e-10, err   # and it falls like dz^4
    # guard: the quantity is sensitive -- shifting the mid-step sample by dz^2 dk'/8 (the difference between the
    # in-step quadratic and a plain average) changes the integral by ~L dz^2 dk'/12 ~ 1e-6 relative
    assert abs(expect) > 0.02 * (2 * np.pi * c["d_eff"] / (c["n2"] * c["lambda1"])) * A0 ** 2 * L


def test_merged_half_steps_equal_unmerged():
    """consecutive linear half-steps are two diagonal factors in the same Fourier basis; applying them as
    one step of length dz (what the fused CUDA path does), with the node powers taken through Parseval, must not
    change anything beyond rounding."""
    w = wl.make("cfg2", nz=24)
    res = []
    for merged in (False, True):
        o = oracle.Oracle(w["grid"], w["crystal"], w["beams"], merged=merged)
        o.set_temperature(w["T"], w["T_uniform"], False)
        a1, a2 = o.propagate(w["A1"].astype(np.complex128), 0.03j * np.roll(w["A1"], 5, axis=2).astype(np.complex128))
        res.append((a1, a2, o.power_history()))
    assert rel_l2(res[1][0], res[0][0]) < 1e-12 and rel_l2(res[1][1], res[0][1]) < 1e-12
    assert np.max(np.abs(res[1][2] / res[0][2] - 1)) < 1e-12
    assert res[0][2][-1, 1] / res[0][2][0, 0] > 1e-3         # light was converted and absorbed on the way
    assert res[0][2][-1].sum() < res[0][2][0].sum() * (1 - 1e-3)


def test_power_lookup_rounds_to_the_nearest_recorded_node():
    """orc_power(z) returns the node nearest to z (powers live on the step nodes z_n = n dz);
    checked at interior and off-node positions against exp(-alpha z_n)."""
    c = wl.crystal(30e-3, d_eff=0.0, alpha1=7.0, alpha2=13.0)
    bm = wl.beam(c, 2.0, 1.5, 12.0)
    n, nz = 16, 10
    A_in = wl.gaussian_pump(n, n, c, bm).astype(np.complex128)
    o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), c, [bm])
    o.propagate(A_in[None], 0.5j * A_in[None])
    h = o.power_history()
    dz = c["L"] / nz
    for z, node in ((0.0, 0), (0.49 * dz, 0), (0.51 * dz, 1), (3.0 * dz, 3), (3.4 * dz, 3), (6.6 * dz, 7),
                    (9.49 * dz, 9), (9.51 * dz, 10), (c["L"], 10), (1.7 * c["L"], 10), (-dz, 0)):
        p1, p2 = o.power(0, z)
        assert abs(p1 / (h[0, 0] * math.exp(-7.0 * node * dz)) - 1) < 1e-12, (z, node)
        assert abs(p2 / (h[0, 1] * math.exp(-13.0 * node * dz)) - 1) < 1e-12, (z, node)


def test_per_member_temperature_and_batch_independence():
    A0, nz, n = 1.0, 128, 4
    g, c, bm, A1 = plane_wave_case(A0, nz, ddk_dT=-30.0)
    dTs = [0.5, 2.0, 3.5]
    T = np.stack([np.full((2, n, n), wl.T_PM + d, np.float32) for d in dTs])
    o = oracle.Oracle(dict(g, nzt=2, batch=3), c, [bm] * 3).set_temperature(T, per_member=True)
    o.propagate(np.repeat(A1, 3, axis=0))
    for b, d in enumerate(dTs):
        h = o.power_history(b)
        assert abs(h[-1, 1] / h[0, 0] / sinc2_expect(c, A0, -30.0 * d) - 1) < 1e-7


# ------------------------------------------------------------------------------------------------
# 7. two-photon absorption: I(z) = I0 / (1 + beta I0 z)   (G5)
# ------------------------------------------------------------------------------------------------
def test_two_photon_absorption_closed_form():
    A0 = 2e7
    g, c, bm, A1 = plane_wave_case(A0, nz=400, d_eff=0.0, beta1=3e-11, beta2=5e-11)
    o = oracle.Oracle(g, c, [bm])
    o.propagate(A1, 0.5 * A1)
    h = o.power_history()
    z = np.linspace(0, c["L"], g["nz"] + 1)
    for j, (beta, nj, amp) in enumerate(((3e-11, c["n1"], A0), (5e-11, c["n2"], 0.5 * A0))):
        I0 = EPS0 * C0 * nj * amp ** 2 / 2
        assert beta * I0 * c["L"] > 0.3                     # strong enough to matter
        assert np.max(np.abs(h[:, j] / h[0, j] * (1 + beta * I0 * z) - 1)) < 1e-10


# ------------------------------------------------------------------------------------------------
# 8. focused SHG in the undepleted limit: Boyd-Kleinman (Eq. 17) with h by quadrature
# ------------------------------------------------------------------------------------------------
def bk_h(sigma, xi):
    """h(sigma, xi) = |int_{-xi}^{xi} e^{i sigma t}/(1 + i t) dt|^2 / (4 xi)  (Boyd & Kleinman 1968, ref. [3]
    of the paper).  The imaginary part of the integrand, (sin(sigma t) - t cos(sigma t))/(1+t^2), is odd,
    so the integral is twice the integral of the even real part over [0, xi]."""
    re = integrate.quad(lambda t: (math.cos(sigma * t) + t * math.sin(sigma * t)) / (1 + t * t), 0.0, xi,
                        epsabs=1e-14, epsrel=1e-13)[0]
    return (2 * re) ** 2 / (4 * xi)


def test_bk_h_function_values():
    assert abs(bk_h(0.0, 2.84) - 0.534654) < 2e-6
    assert abs(bk_h(0.57, 2.84) - 1.067702) < 2e-6
    # "maximum value at xi = 2.84": the optimum over sigma peaks there
    best = {xi: max(bk_h(s, xi) for s in np.linspace(0.3, 0.9, 61)) for xi in (2.0, 2.84, 4.0)}
    assert best[2.84] > best[2.0] and best[2.84] > best[4.0]


@pytest.mark.parametrize("sigma,tol", [(0.0, 1e-4), (0.57, 1e-4), (-0.57, 2e-4)])
def test_focused_shg_matches_boyd_kleinman(sigma, tol):
    xi, P, n, nz = 2.84, 1e-3, 256, 400
    c = wl.crystal(30e-3, n2=2.14)                          # n2 = n1: Eq. 17 assumes k2 = 2 k1 (G26)
    bm = wl.beam(c, P, xi, 30.0)
    b_conf = wl.k1_of(c) * bm["w0"] ** 2
    c["dk0"] = 2 * sigma / b_conf                           # sigma = dk b / 2 (G4)
    A_in = wl.gaussian_pump(n, n, c, bm).astype(np.complex128)
    o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), c, [bm])
    o.propagate(A_in[None])
    h = o.power_history()
    eta = h[-1, 1] / h[0, 0]
    eta_bk = (16 * np.pi ** 2 * c["d_eff"] ** 2 * P * c["L"] /
              (EPS0 * C0 * c["n1"] * c["n2"] * c["lambda1"] ** 3)) * bk_h(sigma, xi)   # Eq. 17
    assert abs(h[0, 0] / P - 1) < 1e-7      # the window holds the whole beam (complex64 input rounding)
    assert abs(eta / eta_bk - 1) < tol


def test_bk_sign_of_mismatch_is_one_sided():
    """the focused-beam optimum sits at non-zero mismatch, on ONE side (Gouy phase): +sigma wins
    by ~48x over -sigma (h = 1.0677 vs 0.0222), so a sign slip in phi, the propagator or Eq. 6 shows."""
    xi, P, n, nz = 2.84, 1e-3, 128, 100
    c = wl.crystal(30e-3, n2=2.14)
    bm = wl.beam(c, P, xi, 24.0)
    b_conf = wl.k1_of(c) * bm["w0"] ** 2
    eta = {}
    for s in (+0.57, -0.57):
        cc = dict(c, dk0=2 * s / b_conf)
        o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), cc, [bm])
        o.propagate(wl.gaussian_pump(n, n, cc, bm).astype(np.complex128)[None])
        h = o.power_history()
        eta[s] = h[-1, 1] / h[0, 0]
    assert 40 < eta[+0.57] / eta[-0.57] < 56
    assert abs(eta[+0.57] / eta[-0.57] / (bk_h(0.57, xi) / bk_h(-0.57, xi)) - 1) < 5e-3


def test_undepleted_switch_and_depleted_deviation():
    """with dPump = 0 the efficiency stays on the BK line; with depletion it falls below it."""
    xi, P, n, nz = 2.84, 20.0, 128, 100
    c = wl.crystal(30e-3, n2=2.14)
    bm = wl.beam(c, P, xi, 24.0)
    A_in = wl.gaussian_pump(n, n, c, bm).astype(np.complex128)[None]
    g = dict(nx=n, ny=n, nz=nz, nzt=0)
    eta_bk = (16 * np.pi ** 2 * c["d_eff"] ** 2 * P * c["L"] /
              (EPS0 * C0 * c["n1"] * c["n2"] * c["lambda1"] ** 3)) * bk_h(0.0, xi)
    o = oracle.Oracle(g, c, [bm], undepleted=True)
    o.propagate(A_in)
    h = o.power_history()
    assert abs(h[-1, 1] / h[0, 0] / eta_bk - 1) < 2e-3
    assert abs(h[-1, 0] / h[0, 0] - 1) < 1e-12              # pump untouched
    o = oracle.Oracle(g, c, [bm])
    o.propagate(A_in)
    h = o.power_history()
    assert h[-1, 1] / h[0, 0] < 0.9 * eta_bk


# ------------------------------------------------------------------------------------------------
# 9. order of the scheme, equivalence of the two orderings
# ------------------------------------------------------------------------------------------------
def test_second_order_convergence_and_ordering_equivalence():
    def run(nz, scheme):
        w = wl.make("cfg1", nz=nz)
        o = oracle.Oracle(w["grid"], w["crystal"], w["beams"], scheme=scheme)
        return o.propagate(w["A1"].astype(np.complex128))[1][0]
    ref = run(3200, 0)
    r0 = {nz: run(nz, 0) for nz in (200, 400, 800)}
    e = [rel_l2(r0[nz], ref) for nz in (200, 400, 800)]
    assert 3.0 < e[0] / e[1] < 8.0 and 3.0 < e[1] / e[2] < 8.0       # global O(dz^2)
    assert abs(e[0] / 2.0e-5 - 1) < 0.1                              # SURVEY.md §8(c) scratch: 2.0e-5 at nz=200
    # the paper's N/2-L-N/2 ordering converges to the same solution ("both lead to the same")
    d = [rel_l2(run(nz, 1), r0[nz]) for nz in (200, 400)]
    assert 2e-5 < d[0] < 6e-5 and 3.0 < d[0] / d[1] < 8.0            # orderings differ 3-4e-5 on CFG1
    assert rel_l2(run(800, 1), ref) < 4 * e[2]


# ------------------------------------------------------------------------------------------------
# 10. symmetry / row-column mix-ups
# ------------------------------------------------------------------------------------------------
def test_radial_symmetry_preserved():
    w = wl.make("cfg1", nz=20)
    o = oracle.Oracle(w["grid"], w["crystal"], w["beams"])
    A1, A2 = o.propagate(w["A1"].astype(np.complex128))
    for A in (A1[0], A2[0]):
        s = np.max(np.abs(A))
        assert np.max(np.abs(A - A.T)) / s < 1e-12
        refl = np.roll(A[::-1, ::-1], (1, 1), axis=(0, 1))            # i -> (N - i) mod N
        assert np.max(np.abs(A - refl)) / s < 1e-12


def test_asymmetric_case_fast_path_equals_definition_path():
    """Off-centre beam, nx != ny, lx != ly, a temperature array that varies in x, y and z, absorption
    and TPA on: the radix-2 path and the brute-force-DFT path must agree (catches any row/column or
    index slip that radial symmetry would hide)."""
    nx, ny, nz = 16, 8, 6
    c = wl.crystal(10e-3, alpha=True, ddk_dT=-300.0)
    c["beta1"] = 2e-11
    w0 = 20e-6
    bm = dict(P=800.0, w0=w0, focus_z=3e-3, lx=9 * w0, ly=6 * w0)
    x, y = wl.axes(nx, ny, bm)
    A_in = wl.gaussian_pump(nx, ny, c, bm).astype(np.complex128)
    A_in = np.roll(A_in, (1, -2), axis=(0, 1)) * np.exp(1j * 2e4 * x)[None, :]
    rng = np.random.default_rng(7)
    T = (wl.T_PM + rng.uniform(0, 3, (4, ny, nx))).astype(np.float32)
    g = dict(nx=nx, ny=ny, nz=nz, nzt=4)
    outs = []
    for brute in (False, True):
        o = oracle.Oracle(g, c, [bm], brute_dft=brute).set_temperature(T)
        outs.append(o.propagate(A_in[None], 0.1 * A_in[None].conj()))
    assert rel_l2(outs[0][0], outs[1][0]) < 1e-12
    assert rel_l2(outs[0][1], outs[1][1]) < 1e-12
    assert np.linalg.norm(outs[0][1]) > 0.05 * np.linalg.norm(outs[0][0])   # strongly coupled case


# ------------------------------------------------------------------------------------------------
# 11. the shared input generator against the oracle's own Eq. 6 (two independent implementations)
# ------------------------------------------------------------------------------------------------
def test_workload_generator_matches_oracle_eq6_and_sizes():
    w = wl.make("cfg1")
    ref = oracle.gaussian_input(w["grid"], w["crystal"], w["beams"][0])
    assert rel_l2(w["A1"][0].astype(np.complex128), ref) < 1e-7           # complex64 rounding only
    assert abs(w["beams"][0]["w0"] - 28.91e-6) < 0.01e-6                  # "w_F = 29 um" at xi = 2.84
    assert wl.algorithmic_bytes_per_point_step(w) == 32.0
    w2 = wl.make("cfg2", nz=10)
    assert w2["T"].shape == (11, 128, 128) and w2["T"].dtype == np.float32
    assert abs(wl.algorithmic_bytes_per_point_step(w2) - (40.0 + 4.0 * 11 / 10)) < 1e-12
    w4 = wl.make("cfg4", nz=4)
    assert len(w4["beams"]) == 64 and w4["A1"].shape == (64, 128, 128)
    assert abs(w4["beams"][0]["w0"] - 108.9e-6) < 0.1e-6 and abs(w4["beams"][63]["w0"] - 15.4e-6) < 0.05e-6


# ------------------------------------------------------------------------------------------------
# 13. heat source of Eq. 8, S§8(f) rank 1: closed forms for its two terms, plane placement (G27),
#     and the energy balance (what the fields lose is what the crystal absorbs)
# ------------------------------------------------------------------------------------------------
def q_steps(nz, nq):
    return [min(nz - 1, ((2 * k + 1) * nz) // (2 * nq)) for k in range(nq)]


def test_heat_source_linear_absorption_closed_form_and_plane_placement():
    A0, a1, a2 = 3e6, 4.0, 9.0
    g, c, bm, A1 = plane_wave_case(A0, nz=60, d_eff=0.0, alpha1=a1, alpha2=a2)
    dz = c["L"] / g["nz"]
    for nq in (60, 7, 1):
        o = oracle.Oracle(g, c, [bm])
        Q = o.set_heat_output(nq)
        o.propagate(A1, 0.5 * A1)
        I1 = EPS0 * C0 * c["n1"] * A0 ** 2 / 2
        I2 = EPS0 * C0 * c["n2"] * (0.5 * A0) ** 2 / 2
        zq = (np.array(q_steps(g["nz"], nq)) + 0.5) * dz           # the sampled mid-step positions
        want = a1 * I1 * np.exp(-a1 * zq) + a2 * I2 * np.exp(-a2 * zq)
        assert Q.shape == (1, nq, g["ny"], g["nx"])
        assert np.max(np.abs(Q[0] / want[:, None, None] - 1)) < 1e-12


def test_heat_source_two_photon_term_closed_form():
    A0, b1, b2 = 2e7, 3e-11, 5e-11
    g, c, bm, A1 = plane_wave_case(A0, nz=400, d_eff=0.0, beta1=b1, beta2=b2)
    dz = c["L"] / g["nz"]
    o = oracle.Oracle(g, c, [bm])
    Q = o.set_heat_output(8)
    o.propagate(A1, 0.5 * A1)
    I1 = EPS0 * C0 * c["n1"] * A0 ** 2 / 2
    I2 = EPS0 * C0 * c["n2"] * (0.5 * A0) ** 2 / 2
    # mean of the source before (I at z_n) and after (I at z_{n+1}) the nonlinear step
    want = 0.0
    for za in (np.array(q_steps(g["nz"], 8)) * dz, (np.array(q_steps(g["nz"], 8)) + 1.0) * dz):
        want = want + 0.5 * (b1 * (I1 / (1 + b1 * I1 * za)) ** 2 + b2 * (I2 / (1 + b2 * I2 * za)) ** 2)
    assert np.max(np.abs(Q[0] / want[:, None, None] - 1)) < 1e-9


def test_heat_source_balances_the_power_the_fields_lose():
    """Focused, converting beam with absorption and TPA: integral of q over the crystal = P(0) - P(L)."""
    c = wl.crystal(20e-3, alpha=True, alpha1=2.0, alpha2=15.0, beta2=4e-11)
    bm = wl.beam(c, 40.0, 1.2, 10.0)
    n, nz = 64, 200
    g = dict(nx=n, ny=n, nz=nz, nzt=0)
    o = oracle.Oracle(g, c, [bm])
    Q = o.set_heat_output(nz)
    o.propagate(wl.gaussian_pump(n, n, c, bm).astype(np.complex128)[None])
    h = o.power_history()
    lost = h[0].sum() - h[-1].sum()
    absorbed = Q.sum() * (bm["lx"] / n) * (bm["ly"] / n) * (c["L"] / nz)
    assert lost / h[0].sum() > 0.05
    assert abs(absorbed / lost - 1) < 2e-5                          # midpoint rule in z, O(dz^2)
    # coarse sampling still integrates a smooth q
    o2 = oracle.Oracle(g, c, [bm])
    Q2 = o2.set_heat_output(25)
    o2.propagate(wl.gaussian_pump(n, n, c, bm).astype(np.complex128)[None])
    assert abs(Q2.sum() * (bm["lx"] / n) * (bm["ly"] / n) * (c["L"] / 25) / lost - 1) < 5e-3


# ------------------------------------------------------------------------------------------------
# 14. spatial walk-off ("tan(rho) dA/dx"; G21): a pure translation by tan(rho) z along x
# ------------------------------------------------------------------------------------------------
def test_walk_off_translates_the_beam_along_x_only():
    c = wl.crystal(20e-3, d_eff=0.0, rho1=0.0, rho2=4e-3)
    bm = wl.beam(c, 1.0, 1.0, 16.0)
    n, nz = 128, 8
    dx = bm["lx"] / n
    # choose rho so that the total shift is a whole number of grid cells: the periodic shift is then exact
    cells = 5
    c["rho2"] = math.atan(cells * dx / c["L"])
    c["rho1"] = math.atan(-2 * dx / c["L"])
    A = wl.gaussian_pump(n, n, c, bm).astype(np.complex128)
    Ain2 = np.roll(A, 7, axis=0) * (0.3 + 0.1j)                    # off-centre in y: a shift in y would show
    ref = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), dict(c, rho1=0.0, rho2=0.0), [bm])
    r1, r2 = ref.propagate(A[None], Ain2[None])
    o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), c, [bm])
    o1, o2 = o.propagate(A[None], Ain2[None])
    s1 = np.linalg.norm(r1)
    assert np.linalg.norm(o2[0] - np.roll(r2[0], cells, axis=1)) / np.linalg.norm(r2) < 1e-11   # SH: +5 cells in x
    assert np.linalg.norm(o1[0] - np.roll(r1[0], -2, axis=1)) / s1 < 1e-11                      # FH: -2 cells
    assert np.linalg.norm(o2[0] - r2[0]) / np.linalg.norm(r2) > 0.1                             # and it did move
    # centroid of a non-integer shift: <x> moves by tan(rho) L
    c2 = dict(c, rho1=1.3e-3, rho2=0.0)
    o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=0), c2, [bm])
    q1, _ = o.propagate(A[None])
    x, _y = wl.axes(n, n, bm)
    cen = lambda a: float((np.abs(a) ** 2 * x[None, :]).sum() / (np.abs(a) ** 2).sum())
    assert abs((cen(q1[0]) - cen(r1[0])) / (math.tan(1.3e-3) * c["L"]) - 1) < 1e-9


# ------------------------------------------------------------------------------------------------
# 15. the COMPLETE path at once (diffraction + walk-off + coupling + depletion + temperature-dependent mismatch +
#     absorption + two-photon absorption) against an independent solver of Eq. 2: method of lines in the
#     interaction picture, numpy FFT, adaptive 8th-order Runge-Kutta (scipy DOP853) at tight tolerance.  Nothing
#     below comes from the oracle: the equations are retyped from the paper with the readings of DESIGN.md §3.
#     The split-step scheme must converge to it at second order in dz.
# ------------------------------------------------------------------------------------------------
def reference_solution(c, bm, n, A1_in, A2_in, Tplanes):
    """A1(L), A2(L) of  dA1/dz = L1 A1 + i kappa1 A2 conj(A1) e^{-i phi} - (beta1/2) I1 A1,
                        dA2/dz = L2 A2 + i kappa2 A1^2 e^{+i phi}        - (beta2/2) I2 A2,
    L_j = -i k_perp^2/(2 k_j) - i kx tan(rho_j) - alpha_j/2 in Fourier space,  I_j = eps0 c n_j |A_j|^2 / 2,
    phi(x,y,z) = int_0^z [dk0 + ddk_dT (T(x,y,z') - T_pm)] dz' with T linear in z between its planes."""
    L = c["L"]
    k1 = 2 * np.pi * c["n1"] / c["lambda1"]
    k2 = 2 * np.pi * c["n2"] / (c["lambda1"] / 2)
    kap1 = 2 * np.pi * c["d_eff"] / (c["n1"] * c["lambda1"])
    kap2 = 2 * np.pi * c["d_eff"] / (c["n2"] * c["lambda1"])
    c1, c2 = EPS0 * C0 * c["n1"] / 2, EPS0 * C0 * c["n2"] / 2
    kx = 2 * np.pi * np.fft.fftfreq(n, d=bm["lx"] / n)[None, :]
    ky = 2 * np.pi * np.fft.fftfreq(n, d=bm["ly"] / n)[:, None]
    kp2 = kx ** 2 + ky ** 2
    lin1 = -1j * kp2 / (2 * k1) - 1j * kx * math.tan(c["rho1"]) - c["alpha1"] / 2
    lin2 = -1j * kp2 / (2 * k2) - 1j * kx * math.tan(c["rho2"]) - c["alpha2"] / 2
    nzt = Tplanes.shape[0]
    zk = np.linspace(0.0, L, nzt)
    dk_k = c["dk0"] + c["ddk_dT"] * (Tplanes.astype(np.float64) - c["T_pm"])         # [nzt][n][n]
    hk = L / (nzt - 1)
    phi_k = np.concatenate([np.zeros((1, n, n)), np.cumsum(0.5 * (dk_k[1:] + dk_k[:-1]) * hk, axis=0)])

    def phi(z):
        k = min(int(z / hk), nzt - 2)
        s = z - zk[k]
        return phi_k[k] + dk_k[k] * s + (dk_k[k + 1] - dk_k[k]) * s * s / (2 * hk)

    def rhs(z, y):
        b1 = y[:n * n].reshape(n, n)
        b2 = y[n * n:].reshape(n, n)
        a1 = np.fft.ifft2(np.exp(lin1 * z) * b1)
        a2 = np.fft.ifft2(np.exp(lin2 * z) * b2)
        e = np.exp(1j * phi(z))
        n1 = 1j * kap1 * a2 * np.conj(a1) / e - 0.5 * c["beta1"] * c1 * np.abs(a1) ** 2 * a1
        n2 = 1j * kap2 * a1 * a1 * e - 0.5 * c["beta2"] * c2 * np.abs(a2) ** 2 * a2
        return np.concatenate([(np.exp(-lin1 * z) * np.fft.fft2(n1)).ravel(), (np.exp(-lin2 * z) * np.fft.fft2(n2)).ravel()])

    y0 = np.concatenate([np.fft.fft2(A1_in).ravel(), np.fft.fft2(A2_in).ravel()])
    scale = np.abs(y0).max()
    sol = integrate.solve_ivp(rhs, (0.0, L), y0, method="DOP853", rtol=1e-11, atol=1e-13 * scale)
    assert sol.success
    y = sol.y[:, -1]
    return (np.fft.ifft2(np.exp(lin1 * L) * y[:n * n].reshape(n, n)),
            np.fft.ifft2(np.exp(lin2 * L) * y[n * n:].reshape(n, n)))


@pytest.mark.parametrize("scheme", [0, 1])
def test_complete_path_converges_to_an_independent_solver_of_eq2(scheme):
    n, nzt = 32, 6
    c = wl.crystal(8e-3, alpha=True, alpha1=3.0, alpha2=20.0, beta1=1e-11, beta2=6e-11, dk0=35.0, ddk_dT=-150.0,
                   rho1=-0.4e-3, rho2=0.9e-3)
    bm = wl.beam(c, 250.0, 1.1, 9.0, focus_z=0.6 * c["L"])
    bm["ly"] = 1.15 * bm["lx"]
    rng = np.random.default_rng(15)
    x, y = wl.axes(n, n, bm)
    A1 = np.roll(wl.gaussian_pump(n, n, c, bm), (2, -1), axis=(0, 1)).astype(np.complex128)
    A2 = 0.05 * np.roll(A1, 3, axis=1) * np.exp(0.4j)
    # smooth asymmetric temperature planes (the mismatch phase varies by several rad across the beam and along z)
    T = np.empty((nzt, n, n), dtype=np.float32)
    for k in range(nzt):
        T[k] = (wl.T_PM + 1.5 * np.exp(-((x[None, :] - 0.2 * bm["w0"]) ** 2 + (y[:, None] + 0.1 * bm["w0"]) ** 2)
                                       / (1.5 * bm["w0"]) ** 2) * (0.3 + 0.2 * k) + 0.05 * rng.standard_normal())
    r1, r2 = reference_solution(c, bm, n, A1, A2, T)
    assert np.linalg.norm(r2) / np.linalg.norm(r1) > 0.15          # a strongly converting, depleting case
    errs = []
    sols = []
    for nz in (40, 80, 160):                                        # plane knots sit on step nodes (5 divides nz)
        o = oracle.Oracle(dict(nx=n, ny=n, nz=nz, nzt=nzt), c, [bm], scheme=scheme)
        o.set_temperature(T, 0.0, False)
        o1, o2 = o.propagate(A1[None], A2[None])
        sols.append((o1[0], o2[0]))
        errs.append((rel_l2(o1[0], r1), rel_l2(o2[0], r2)))
    for j in (0, 1):
        assert 3.5 < errs[0][j] / errs[1][j] < 4.5 and 3.5 < errs[1][j] / errs[2][j] < 4.5, errs   # second order
        assert errs[2][j] < 3e-5, errs
    # Richardson extrapolation of the two finest runs removes the dz^2 term: what is left is the oracle's own error
    e1 = (4 * sols[2][0] - sols[1][0]) / 3
    e2 = (4 * sols[2][1] - sols[1][1]) / 3
    assert rel_l2(e1, r1) < 5e-8 and rel_l2(e2, r2) < 5e-8, (rel_l2(e1, r1), rel_l2(e2, r2))   # measured 3e-9, 6e-9
