"""tdh_overlap_noalloc: the overlap matrix for callers that must not allocate device memory.

Some users of this library cannot call cudaMalloc where they need an overlap matrix: a simulation code whose own pool
has taken the device's memory (the paper's code keeps such a pool so that hot paths never allocate), a
propagation loop that must not be stalled by an allocation's device-wide synchronisation, or a tool that only wants to
check orthonormality and will not create a tdh_grid with its gigabytes of workspace for that.  For them the library has
one entry point whose split-K scratch is a fixed 8 MiB array inside libtdh.so (limit: 256 x 256 states).  Every call
shares that array and finds the previous call's partial tiles in it, so the tests below always make two calls in a
row, with different shapes, and compare BOTH with the existing handle-based path (tdh_overlap, workspace scratch) at
the tolerance of the other overlap tests (1e-13 of the Cauchy-Schwarz scale; the two paths may cut K into a different
number of slices, so they agree to rounding, not bitwise).

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this extra entry point
must not hide the parity tests of the hot path.  It depends on nothing the other test files leave behind and passes in a
fresh process as well as after them.
"""
import numpy as np
import pytest

from paper_2106_03872_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-13


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device: the product has no CPU fallback")
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2106_03872_b200 import binding
    binding.lib()
    return binding


def blocks(n, na, nb, tag):
    rng = np.random.default_rng([W.BASE_SEED, 77, na, nb, tag])
    a = rng.standard_normal((na,) + n) + 1j * rng.standard_normal((na,) + n)
    b = rng.standard_normal((nb,) + n) + 1j * rng.standard_normal((nb,) + n)
    return a, b


def cs_scale(a, b, dv):
    """Largest |a_i| |b_j| dV: the size an overlap element can reach (Cauchy-Schwarz)."""
    ax = tuple(range(1, a.ndim))
    return float(np.sqrt(np.outer(np.sum(np.abs(a) ** 2, axis=ax), np.sum(np.abs(b) ** 2, axis=ax))).max() * dv)


def test_two_calls_in_a_row_match_the_handle_path(torch_cuda, B):
    """Call 1 fills most of the scratch array (256 x 200 states, several slices of K); call 2 is a small ragged block on
    another grid and must not see any of it; call 3 is one block against itself (upper tiles + mirror).  Each result is
    compared with tdh_overlap of a handle."""
    torch = torch_cuda
    cases = [((32, 16, 48), 256, 200, False), ((16, 48, 16), 5, 70, False), ((32, 32, 16), 130, 130, True)]
    got, want, scales = [], [], []
    dev = []
    for tag, (n, na, nb, same) in enumerate(cases):
        a, b = blocks(n, na, nb, tag)
        length = tuple(0.5 * m for m in n)
        dv = float(np.prod([length[i] / n[i] for i in range(3)]))
        da = torch.from_numpy(a).cuda()
        db = da if same else torch.from_numpy(b).cuda()
        dev.append((n, length, dv, da, db))
        scales.append(cs_scale(a, a if same else b, dv))
    # the new entry point, back to back on one stream, outputs preallocated: nothing but the launches in between
    outs = [torch.empty((c[1], c[2]), dtype=torch.complex128, device="cuda") for c in cases]
    for (n, length, dv, da, db), out in zip(dev, outs):
        B.overlap_noalloc(da, db, dv=dv, out=out)
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in outs]
    for (n, length, dv, da, db), (_, na, nb, _) in zip(dev, cases):
        with B.Grid(n, length, (0.0, 0.0, 0.0), -1.0, max(na, nb)) as g:
            want.append(g.overlap(da, db).cpu().numpy())
    for s_new, s_old, scale, case in zip(got, want, scales, cases):
        assert s_new.shape == s_old.shape
        assert np.abs(s_new - s_old).max() <= TOL * scale, case
    # the same first call again, after the others have overwritten the array: the same bits as before
    again = B.overlap_noalloc(dev[0][3], dev[0][4], dv=dev[0][2]).cpu().numpy()
    assert np.array_equal(again, got[0])
    herm = got[2]
    assert np.abs(herm - herm.conj().T).max() <= TOL * scales[2]


def test_ragged_point_count_and_plain_product(torch_cuda, B):
    """No divisibility requirement on the number of points (the handle path needs a multiple of 64): 7 x 5 x 9 = 315
    points, dv = 1, against the product written out with torch on the device; twice in a row with swapped operands."""
    torch = torch_cuda
    n = (7, 5, 9)
    a, b = blocks(n, 3, 67, 9)
    da, db = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    s_ab = B.overlap_noalloc(da, db)
    s_ba = B.overlap_noalloc(db, da)
    ref = a.reshape(3, -1).conj() @ b.reshape(67, -1).T
    scale = cs_scale(a, b, 1.0)
    assert np.abs(s_ab.cpu().numpy() - ref).max() <= TOL * scale
    assert np.abs(s_ba.cpu().numpy() - ref.conj().T).max() <= TOL * scale


def test_sizes_beyond_the_fixed_scratch_are_refused(torch_cuda, B):
    """257 states do not fit the array's layout: a clear error, and the next call in range still works."""
    torch = torch_cuda
    assert B.NOALLOC_MAX_STATES == 256
    big = torch.zeros((257, 64), dtype=torch.complex128, device="cuda")
    small = torch.ones((2, 64), dtype=torch.complex128, device="cuda")
    for x, y in ((big, small), (small, big)):
        with pytest.raises(B.TdhError) as err:
            B.overlap_noalloc(x, y)
        assert err.value.code == B.TDH_EUNSUPPORTED
        assert "256" in str(err.value) and "tdh_overlap" in str(err.value)
    s = B.overlap_noalloc(small, small, dv=0.5).cpu().numpy()
    assert np.array_equal(s, np.full((2, 2), 32.0 + 0.0j))
