"""The GPU's own Philox4x32-10 words (the generator inside k_step / k_sweep_small, exposed as qmc_philox_words), checked
directly: against the published known-answer vectors, against the oracle's generator, and against cuRAND's device
Philox4x32-10 -- an implementation that shares nothing with either (second pin of row 1)."""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

qb = pytest.importorskip("paper_2504_07948_b200")
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    qb.load_library()


def _inputs(n, seed):
    rng = np.random.default_rng(seed)
    ck = rng.integers(0, 2 ** 32, size=(n, 6), dtype=np.uint64).astype(np.uint32)
    ck[:, 1] &= 0x3FFFFFFF          # cuRAND takes the low counter pair as offset / 4: keep 4 * (c1 c0) inside 64 bits
    ck[: n // 4, 1] = np.arange(n // 4) % 50                     # the values a run really uses: small sweep counters,
    ck[: n // 4, 2] = rng.integers(0, 4096, n // 4)              # electron indices,
    ck[: n // 4, 3] = np.arange(n // 4) % 6                      # block numbers 0..5
    return ck


def test_known_answer_vectors_on_the_gpu():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    ck = np.array([[int(x, 16) for x in r[:6]] for r in rows], np.uint32)
    want = np.array([[int(x, 16) for x in r[6:10]] for r in rows], np.uint32)
    assert np.array_equal(qb.qmc_philox_words(ck), want)


def test_gpu_words_equal_the_oracles():
    ck = _inputs(2048, 1)
    got = qb.qmc_philox_words(ck)
    for i in range(0, 2048, 7):
        assert np.array_equal(got[i], oracle.philox4x32_10(ck[i, :4], ck[i, 4:]))


def test_gpu_words_equal_curand_device_philox():
    nvcc = os.environ.get("NVCC") or shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("no nvcc to build the cuRAND helper")
    out_dir = os.path.join(HERE, "cuda", "_build")
    os.makedirs(out_dir, exist_ok=True)
    lib_path = os.path.join(out_dir, "libcurand_philox_ref.so")
    src = os.path.join(HERE, "cuda", "curand_philox_ref.cu")
    if not os.path.exists(lib_path) or os.path.getmtime(lib_path) < os.path.getmtime(src):
        subprocess.run([nvcc, "-O2", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-shared", "-o", lib_path, src],
                       check=True, capture_output=True)
    ref = C.CDLL(lib_path)
    ref.curand_philox_words.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    ck = _inputs(8192, 2)
    want = np.zeros((len(ck), 4), np.uint32)
    assert ref.curand_philox_words(len(ck), ck.ctypes.data, want.ctypes.data) == 0
    got = qb.qmc_philox_words(ck)
    assert np.array_equal(got, want)
    assert len(np.unique(got)) > 0.99 * got.size     # (not all equal by being all zero)
