"""sg_chiral_cross_static, the entry point that allocates nothing, against sg_chiral_cross (the existing path).

Why the entry point exists: some users of this library hold two zeta buffers on the device and want their chiral-glass
overlaps (Eq. (2)) from a place where no allocating call may be made -- a measurement process on a GPU whose
memory the Monte Carlo workspaces (or a framework's pool) already own in full, a loop where the device-wide stall of
cudaMalloc / cudaFree would stop the sweeps on the other streams, or host code that is not allowed near the allocator.  They
have no sg_ctx (a context pins host memory and needs a workspace); the partial sums therefore live in a fixed 16 MiB array
inside the library, shared by every call on the device and never cleared.

What is checked here: the new call reproduces the existing one within 1e-12 (the bar tests/test_gpu_observables.py holds the
cross-context overlaps to; the two differ only in the last bit of the Fourier phase table) on consecutive calls -- including
a call with a SMALLER shape after a larger one and back, so that the leftovers in the shared array would show if any element
were read before being written -- that the driver's free-memory figure does not move across a call, and that a shape beyond
the array is refused with SG_ELIMIT instead of being served some other way.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It has no dependence on what ran before it (alone in a fresh process the first call below is also the first
use of the array on the device; after the other tests the library is merely already loaded)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


def make(sg, L, S, T, seed):
    g = sg.SpinGlass(L, S, 2, T, np.linspace(0.5, 2.0, T), seed=seed)
    for s in range(S):
        g.init_sample(s)
    for _ in range(2):
        g.unit(2)
    return g


def both_paths(sg, g, out=None):
    """(existing path, new entry point) for the replica pair (0, 1) of context g, as host arrays."""
    import torch
    za, zb = g.export_chirality(0), g.export_chirality(1)
    qc0_ref, qck_ref = g.chiral_cross(za, zb)                       # existing path: partial sums in the context's workspace
    qc0, qck = sg.chiral_cross_static(g.L, g.S, g.T, za, zb, out=out)     # new: partial sums in the library's fixed array
    torch.cuda.synchronize()
    return (qc0_ref, qck_ref), (qc0.cpu().numpy(), qck.cpu().numpy())


def test_static_entry_point_matches_the_existing_path_on_consecutive_calls(sg):
    import torch
    big = make(sg, 8, 3, 16, seed=5)        # 3 samples: the most the array is guaranteed to take
    small = make(sg, 6, 2, 10, seed=6)      # fewer samples, ragged site chunks (216 sites over 128 chunks), other T
    seen = []
    for g in (big, small, big, big):        # larger -> smaller -> larger again -> same shape twice in a row
        (r0, rk), (q0, qk) = both_paths(sg, g)
        assert q0.shape == r0.shape and qk.shape == rk.shape
        assert np.isfinite(q0).all() and np.isfinite(qk).all()
        assert np.abs(q0 - r0).max() <= TOL and np.abs(qk - rk).max() <= TOL, (np.abs(q0 - r0).max(), np.abs(qk - rk).max())
        assert np.abs(r0).max() > 1e-4                                # a real signal, not zeros against zeros
        seen.append(q0.copy())
        g.unit(2)                                                     # the next call sees other spins
    assert np.abs(seen[2] - seen[0]).max() > 1e-6 and np.abs(seen[3] - seen[2]).max() > 1e-6
    # same inputs twice in a row give the same bits (nothing carried over from call to call)
    za, zb = big.export_chirality(0), big.export_chirality(1)
    a = torch.cat([t.reshape(-1) for t in sg.chiral_cross_static(big.L, big.S, big.T, za, zb)]).clone()
    b = torch.cat([t.reshape(-1) for t in sg.chiral_cross_static(big.L, big.S, big.T, za, zb)]).clone()
    assert torch.equal(a, b)
    for g in (big, small):
        g.close()


def test_static_entry_point_leaves_device_memory_alone_and_refuses_oversized_shapes(sg):
    import torch
    g = make(sg, 8, 2, 12, seed=9)
    za, zb = g.export_chirality(0), g.export_chirality(1)
    out = torch.empty(g.S * g.T * 21, dtype=torch.float64, device=za.device)
    ref0, refk = g.chiral_cross(za, zb)
    sg.chiral_cross_static(g.L, g.S, g.T, za, zb, out=out)            # set-up call (first on this device if run alone)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                        # the driver's figure, not torch's pool
    for _ in range(2):
        q0, qk = sg.chiral_cross_static(g.L, g.S, g.T, za, zb, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert q0.data_ptr() == out.data_ptr()                            # the caller's buffer, no copy
    assert np.abs(q0.cpu().numpy() - ref0).max() <= TOL and np.abs(qk.cpu().numpy() - refk).max() <= TOL
    # 4 samples x 12 temperatures need 4096 + 4 * 128 * 252 * 168 bytes = 20.7 MiB > 16 MiB: refused, output untouched
    S_big = 4
    zz = torch.zeros((S_big, 3, g.N, g.T), dtype=torch.float32, device=za.device)
    sentinel = torch.full((S_big * g.T * 21,), 123.0, dtype=torch.float64, device=za.device)
    with pytest.raises(sg.SgError) as info:
        sg.chiral_cross_static(g.L, S_big, g.T, zz, zz, out=sentinel)
    assert info.value.code == sg.SG_ELIMIT and "SG_STATIC_SCRATCH_BYTES" in str(info.value)
    torch.cuda.synchronize()
    assert bool((sentinel == 123.0).all())
    # ... and the caller's way out: one call per group of <= 3 samples on one stream gives the whole answer
    g4 = make(sg, 6, 4, 12, seed=11)
    za4, zb4 = g4.export_chirality(0), g4.export_chirality(1)
    ref0, refk = g4.chiral_cross(za4, zb4)
    q0a, qka = sg.chiral_cross_static(g4.L, 3, g4.T, za4[:3], zb4[:3])
    q0b, qkb = sg.chiral_cross_static(g4.L, 1, g4.T, za4[3:], zb4[3:])
    torch.cuda.synchronize()
    # the second call reused the array the first one had filled: its result must have been read out in stream order
    q0 = torch.cat([q0a, q0b]).cpu().numpy(); qk = torch.cat([qka, qkb]).cpu().numpy()
    assert np.abs(q0 - ref0).max() <= TOL and np.abs(qk - refk).max() <= TOL
    g.close(); g4.close()
