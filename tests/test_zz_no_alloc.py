"""qmc_eval_basis_noalloc (include/qmc.h): the basis kernel with its scratch -- the pre-tiled A operand -- in a fixed
`static __device__` array of the library, for callers that may not allocate device memory.  Its output is checked against
the existing, allocating qmc_eval_basis on two calls in a row (the second with fewer points and other positions, so that
anything left in the shared array by the first call would show).  Collected last on purpose (the suite runs with
pytest -x)."""
import numpy as np
import pytest

import qmc_inputs as qi

pytestmark = pytest.mark.gpu

qb = pytest.importorskip("paper_2504_07948_b200")

REL_TOL = 1e-13     # the tolerance of test_gpu_parity.test_basis_and_mo_rows for these rows


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    qb.load_library()
    return torch


def _points(s, n, seed):
    rng = np.random.default_rng(seed)
    return s.atoms_xyz[rng.integers(0, s.n_atoms, n)] + rng.standard_normal((n, 3)) * 1.2


@pytest.mark.parametrize("cfg,n_first,n_second", [(0, 300, 41), (1, 70, 9)])
def test_noalloc_basis_equals_the_allocating_path_twice_in_a_row(torch_cuda, cfg, n_first, n_second):
    torch = torch_cuda
    s = qi.make_system(cfg)
    g = qb.qmc_init_from(s)
    for call, n in enumerate((n_first, n_second)):
        pts = _points(s, n, 100 * cfg + call)
        want = qb.qmc_eval_basis(g, pts).cpu().numpy()                        # existing path: allocates its scratch per call
        xyz = torch.from_numpy(pts).cuda()
        out = torch.full((n, 5, s.n_basis), float("nan"), dtype=torch.float64, device="cuda")   # the caller's output buffer
        qb.qmc_eval_basis_noalloc(g, xyz, out)
        torch.cuda.current_stream().synchronize()                              # the call only enqueues
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        assert np.abs(got - want).max() <= REL_TOL * np.abs(want).max(), (cfg, call)
        assert np.abs(want).max() > 1e-3


def test_noalloc_rejects_sizes_beyond_the_fixed_array_and_host_pointers(torch_cuda):
    torch = torch_cuda
    s = qi.make_system(1)
    g = qb.qmc_init_from(s)
    kb = (s.n_basis + 31) // 32
    max_points = (8 << 20) // (128 * 36 * 8 * kb) * 128 // 5                     # the limit stated in include/qmc.h
    for n, ok in ((max_points, True), (max_points + 1, False)):
        xyz = torch.from_numpy(_points(s, n, 7)).cuda()
        out = torch.empty((n, 5, s.n_basis), dtype=torch.float64, device="cuda")
        if ok:
            qb.qmc_eval_basis_noalloc(g, xyz, out)
            torch.cuda.current_stream().synchronize()
            want = qb.qmc_eval_basis(g, xyz).cpu().numpy()
            assert np.abs(out.cpu().numpy() - want).max() <= REL_TOL * np.abs(want).max()
        else:
            with pytest.raises(qb.QmcError, match=f"at most {max_points} points"):
                qb.qmc_eval_basis_noalloc(g, xyz, out)
    # host memory is not accepted (the ABI is called directly: the binding would refuse a numpy array itself)
    import ctypes as C
    pts = np.ascontiguousarray(_points(s, 4, 8))
    out = torch.empty((4, 5, s.n_basis), dtype=torch.float64, device="cuda")
    lib = qb.load_library()
    rc = lib.qmc_eval_basis_noalloc(g.handle, 4, C.c_void_p(pts.ctypes.data), C.c_void_p(out.data_ptr()), None)
    assert rc != 0 and b"device memory" in lib.qmc_last_error()
