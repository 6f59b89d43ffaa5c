"""shg_field_power_static, the entry point for callers that cannot allocate, against the existing path.

Some users of a power integral may not call cudaMalloc at all: code that runs inside another allocator or memory
pool, a plug-in whose host application owns every byte of device memory, a loop that cannot take the driver's
allocation lock.  They cannot create a libshg context (shg_create allocates), so include/shg.h gives them one call
that needs none and keeps its scratch in a fixed array inside the library.  This test checks that call against what
the context-based path reports for the same fields: shg_propagate sums the power of its inputs (k_input_power) and
shg_power_history returns it as node 0.

Two calls in a row, on different shapes, so that the second one runs on the array as the first one left it.  The
file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests), and
it passes alone in a fresh process as well as after everything else: it depends on nothing the other tests leave
behind, and the library clears the part of its scratch that must start at zero on every call.

Tolerance.  Both paths add the same chunks in double in the same order, so the sums agree exactly; the existing path
then stores them in fixed point scaled so that P1 + P2 fills 56 bits (shg_device.cuh, "power sums"), which rounds
each field's sum by at most 2^-56 of the total.  1e-12 of the total input power covers that and the one
multiplication by the scale, and is far inside the 1e-4 the parity tests allow on powers.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2410_04994_b200 import shg
from paper_2410_04994_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_OF_TOTAL = 1e-12


def _scales(w, b):
    """(eps0 c n_j / 2) dx dy of member b: what turns sum |A_j|^2 into W."""
    g, c, bm = w["grid"], w["crystal"], w["beams"][b]
    cell = (bm["lx"] / g["nx"]) * (bm["ly"] / g["ny"])
    return [0.5 * wl.EPS0 * wl.C0 * c[n] * cell for n in ("n1", "n2")]


def _existing_path(w, A1, A2):
    """P_j(0) of every member as the context-based path reports it (shg_propagate + shg_power_history)."""
    ctx = shg.Shg(w["grid"], w["crystal"], w["beams"])
    if w["grid"]["nzt"] > 0:
        T = torch.from_numpy(w["T"]).cuda()
        ctx.set_temperature(T, per_member=w["per_member"])
    else:
        ctx.set_temperature(None, w["T_uniform"])
    ctx.propagate(A1, A2)
    ref = np.stack([ctx.power_history(b)[0] for b in range(A1.shape[0])])
    ctx.close()
    return ref


def _case(name, nz, sh_seed):
    w = wl.make(name, nz=nz)
    g = w["grid"]
    A1 = torch.from_numpy(w["A1"]).cuda().reshape(-1, g["ny"], g["nx"])
    rms = float(np.sqrt(np.mean(np.abs(w["A1"]) ** 2)))
    A2 = torch.from_numpy(wl.noisy_sh_seed(g["nx"], g["ny"], 0.3 * rms, sh_seed, batch=A1.shape[0])).cuda()
    return w, A1, A2.reshape(A1.shape)


def _static_path(w, A1, A2, out):
    """The same numbers from shg_field_power_static.  The members of a sweep have their own windows, hence their own
    scale: the call takes one scale per field, so it is given 1 and the per-member factor is applied to its sums."""
    shg.field_power_static(A1, A2, 1.0, 1.0, out)
    torch.cuda.synchronize()
    sums = out.cpu().numpy().reshape(-1, 2)
    return np.stack([sums[b] * np.array(_scales(w, b)) for b in range(sums.shape[0])])


def test_static_scratch_power_matches_context_path_on_two_calls_in_a_row():
    # first call: the 8 x 8 sweep (64 members of 128 x 128, four chunk sums each);
    # second call: one 256 x 256 simulation (16 chunk sums) -- fewer members, more chunks, same scratch
    cases = [_case("cfg4", 2, 11), _case("cfg3", 2, 12)]
    refs = [_existing_path(*c) for c in cases]
    outs = [torch.full((c[1].shape[0], 2), float("nan"), dtype=torch.float64, device="cuda") for c in cases]
    # set-up call: the first call on a device looks the scratch array up (and may make the CUDA runtime load the
    # library's device image); include/shg.h asks for it to be made during set-up.  From here on nothing may allocate.
    shg.field_power_static(cases[1][1], None, 1.0, 1.0, outs[1])
    torch.cuda.synchronize()
    outs[1].fill_(float("nan"))
    free_before = torch.cuda.mem_get_info()[0]
    got = [_static_path(w, A1, A2, out) for (w, A1, A2), out in zip(cases, outs)]
    assert torch.cuda.mem_get_info()[0] == free_before, "the static path took device memory"
    for (w, A1, A2), ref, val in zip(cases, refs, got):
        assert val.shape == ref.shape and np.all(np.isfinite(val))
        assert np.all(val[:, 1] > 0), "the SH seed carries power"
        total = ref.sum(axis=1, keepdims=True)
        assert np.all(np.abs(val - ref) <= TOL_OF_TOTAL * total), (w["name"], np.max(np.abs(val - ref) / total))

    # once more on the first shape: the array now holds the second call's leftovers; same bits as before
    w, A1, A2 = cases[0]
    again = _static_path(w, A1, A2, outs[0])
    assert np.array_equal(again, got[0])

    # no second harmonic: P2 = 0, P1 unchanged; a scale given to the call is applied by the kernel
    s1, s2 = _scales(w, 0)
    shg.field_power_static(A1[:1], None, s1, s2, outs[0][:1])
    torch.cuda.synchronize()
    p = outs[0][0].cpu().numpy()
    assert p[1] == 0.0 and abs(p[0] - refs[0][0, 0]) <= TOL_OF_TOTAL * refs[0][0].sum()


def test_static_scratch_limit_is_an_error_not_an_overrun():
    n = shg.STATIC_MAX_BATCH + 1
    A = torch.zeros((n, 4, 4), dtype=torch.complex64, device="cuda")
    out = torch.full((n, 2), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(shg.ShgError) as err:
        shg.field_power_static(A, None, 1.0, 1.0, out)
    assert err.value.code == shg.SHG_ELIMIT and "SHG_STATIC_MAX_BATCH" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == -1.0).all()), "a rejected call must not touch its output"
    # the largest size that is allowed, on a ragged grid (no power of two, chunk tail shorter than the rest)
    A = torch.randn((shg.STATIC_MAX_BATCH, 70, 130, 2), device="cuda").contiguous()
    Ac = torch.view_as_complex(A)
    shg.field_power_static(Ac, None, 1.0, 1.0, out[:-1])
    torch.cuda.synchronize()
    want = (A.double() ** 2).sum(dim=(1, 2, 3)).cpu().numpy()
    got = out[:-1, 0].cpu().numpy()
    assert np.all(np.abs(got - want) <= 1e-12 * want) and bool((out[:-1, 1] == 0).all())
