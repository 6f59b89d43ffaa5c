"""Seeded random sweep of the CUDA path against the oracle: grid sizes (square and rectangular), z-step counts,
every temperature encoding, per-member arrays, batches, SH seeds, walk-off, FH two-photon absorption, both
orderings of the split step, the undepleted switch, heat output, both launch schemes -- in combinations the
hand-written cases of test_gpu_parity.py do not enumerate."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2410_04994_b200 import shg
from paper_2410_04994_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SIZES = [64, 128, 256, 512]


def rel(a, b):
    nb = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (nb if nb > 0 else 1.0))


@pytest.mark.parametrize("seed,pipe", [(11, False), (12, False), (13, False), (21, True), (22, True)])
def test_random_configurations_match_oracle(seed, pipe):
    """pipe: the same draws bent to batches of square grids in the pipelined batched kernel (SHG_OPT_PIPELINE = 2),
    half of them with the temperature array handed over as a HOST array."""
    rng = np.random.default_rng(seed)
    for case in range(10):
        nx = int(rng.choice(SIZES, p=[0.35, 0.35, 0.2, 0.1]))
        ny = nx if rng.random() < 0.6 else int(rng.choice(SIZES, p=[0.35, 0.35, 0.2, 0.1]))
        nz = int(rng.integers(2, 13))
        batch = int(rng.integers(1, 4)) if nx * ny <= 256 * 256 else 1
        nzt = int(rng.choice([0, 1, 2, 3, nz + 1, 5]))
        per_member = bool(rng.random() < 0.4) and nzt > 0 and batch > 1
        scheme = int(rng.random() < 0.3)
        undep = bool(rng.random() < 0.2)
        persistent = bool(rng.random() < 0.6)
        nq = int(rng.integers(1, nz + 1)) if (rng.random() < 0.35 and scheme == 0) else 0
        host_T = False
        if pipe:
            ny, scheme, nq, persistent = nx, 0, 0, True
            batch = int(rng.integers(2, 6)) if nx <= 256 else 2
            per_member = bool(rng.random() < 0.5) and nzt > 0
            host_T = bool(rng.random() < 0.5)
        c = wl.crystal(float(rng.uniform(4e-3, 12e-3)), alpha=True, ddk_dT=float(rng.uniform(-400, 400)),
                       dk0=float(rng.uniform(-50, 50)), beta1=float(rng.choice([0.0, 2e-11])),
                       rho1=float(rng.choice([0.0, 1e-3])), rho2=float(rng.choice([0.0, -2e-3])))
        beams = [wl.beam(c, float(rng.uniform(1, 60)), float(rng.uniform(0.3, 3)), float(rng.uniform(6, 12)),
                         focus_z=float(rng.uniform(0, 1)) * c["L"]) for _ in range(batch)]
        for bm in beams:
            bm["ly"] = bm["lx"] * float(rng.uniform(0.7, 1.4))
        g = dict(nx=nx, ny=ny, nz=nz, nzt=nzt, batch=batch)
        A1 = np.stack([np.roll(wl.gaussian_pump(nx, ny, c, bm), (int(rng.integers(-5, 6)), int(rng.integers(-5, 6))),
                               axis=(0, 1)) for bm in beams])
        A2 = (0.1 * np.roll(A1, 3, axis=2) * np.exp(0.7j)).astype(np.complex64) if rng.random() < 0.5 else None
        Tu = wl.T_PM + float(rng.uniform(-1, 1))
        T = None
        if nzt > 0:
            T = (wl.T_PM + rng.uniform(-2, 2, size=((batch if per_member else 1), nzt, ny, nx))).astype(np.float32)
        tag = ("seed %d case %d: %dx%d nz %d batch %d nzt %d per_member %d scheme %d undepleted %d persistent %d nq %d"
               % (seed, case, nx, ny, nz, batch, nzt, per_member, scheme, undep, persistent, nq))

        ctx = shg.Shg(g, c, beams, persistent=persistent)
        ctx.set_option(shg.OPT_SCHEME, scheme)
        ctx.set_option(shg.OPT_UNDEPLETED, int(undep))
        if pipe:
            ctx.set_option(shg.OPT_PIPELINE, 2)
            ctx.set_option(shg.OPT_CLUSTER, 0)
        if nzt > 0:
            Td = T if host_T else torch.from_numpy(T).cuda()
            ctx.set_temperature(Td, per_member=per_member)
        else:
            ctx.set_temperature(None, Tu)
        Q = None
        if nq:
            Q = torch.full((batch, nq, ny, nx), float("nan"), dtype=torch.float32, device="cuda")
            ctx.set_heat_output(Q)
        g1, g2 = ctx.propagate(torch.from_numpy(A1).cuda(), None if A2 is None else torch.from_numpy(A2).cuda())
        torch.cuda.synchronize()
        if pipe:
            assert ctx.last_kernel() == 3, tag

        o = oracle.Oracle(g, c, beams, scheme=scheme, undepleted=undep)
        o.set_temperature(T, Tu, per_member)
        Qo = o.set_heat_output(nq) if nq else None
        o1, o2 = o.propagate(A1.astype(np.complex128), None if A2 is None else A2.astype(np.complex128))
        for b in range(batch):
            assert rel(g1.cpu().numpy()[b], o1[b]) <= 2e-5, tag
            assert rel(g2.cpu().numpy()[b], o2[b]) <= 2e-5, tag
            ho = o.power_history(b)
            assert np.max(np.abs(ctx.power_history(b) - ho)) / ho.max() <= 2e-5, tag
            if nq:
                Qg = Q.cpu().numpy().astype(np.float64)
                assert np.isfinite(Qg).all() and rel(Qg[b], Qo[b]) <= 2e-5, tag
        ctx.close()
        o.close()
