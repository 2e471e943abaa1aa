"""Pins for the oracle's Philox4x32-10 and uniform mapping (no GPU)."""
import ctypes as C
import numpy as np
import pytest

from oracle import philox4x32_10, u01


def _curand_host():
    for name in ("libcurand.so.10", "libcurand.so", "/usr/local/cuda/lib64/libcurand.so.10",
                 "/usr/local/cuda/lib64/libcurand.so"):
        try:
            return C.CDLL(name)
        except OSError:
            continue
    return None


def test_against_curand_host_generator():
    """cuRAND's HOST Philox4x32-10 generator runs on the CPU.  With the default
    ordering its 4-word block j is Philox(counter=(j>>16, 0, j&0xFFFF, 0), key=seed)
    (mapping found by search); every block must equal ours."""
    lib = _curand_host()
    if lib is None:
        pytest.fail("libcurand (CUDA toolkit) not loadable: the Philox pin needs it")
    gen = C.c_void_p()
    CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    if lib.curandCreateGeneratorHost(C.byref(gen), CURAND_RNG_PSEUDO_PHILOX4_32_10) != 0:
        pytest.fail("cuRAND host generator unavailable: the Philox pin needs it")
    for seed in (0, 77, 0x0123456789ABCDEF):
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(gen, C.c_ulonglong(0)) == 0
        nblk = 70000
        out = np.zeros(4 * nblk, np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(out.size)) == 0
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for j in list(range(0, 40)) + [4095, 4096, 65535, 65536, 65537, 69999]:
            got = philox4x32_10((j >> 16, 0, j & 0xFFFF, 0), key)
            assert got == tuple(int(x) for x in out[4 * j:4 * j + 4]), (seed, j)
    lib.curandDestroyGenerator(gen)


def test_counter_words_are_all_used():
    base = philox4x32_10((1, 2, 3, 4), (5, 6))
    for k in range(4):
        c = [1, 2, 3, 4]
        c[k] += 1
        assert philox4x32_10(c, (5, 6)) != base
    assert philox4x32_10((1, 2, 3, 4), (6, 6)) != base
    assert philox4x32_10((1, 2, 3, 4), (5, 7)) != base
    assert philox4x32_10((2, 1, 3, 4), (5, 6)) != base      # not symmetric in the counter


def test_uniform_mapping_exact_in_fp32_and_open_interval():
    xs = [0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 0xFFFFFE00]
    for x in xs:
        u = u01(x)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                      # representable in fp32
        assert u == ((x >> 9) + 0.5) / 2 ** 23
    assert u01(0) == 2.0 ** -24 and u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24


def test_uniformity_smoke():
    w = np.array([philox4x32_10((i, 0, 1, 2), (0, 0)) for i in range(4000)], dtype=np.uint64)
    u = ((w >> 9).astype(np.float64) + 0.5) / 2 ** 23
    assert abs(u.mean() - 0.5) < 4 / np.sqrt(12 * u.size)
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.08
    hist, _ = np.histogram(u.ravel(), bins=16, range=(0, 1))
    chi2 = ((hist - u.size / 16) ** 2 / (u.size / 16)).sum()
    assert chi2 < 45.0                                        # 15 dof, p ~ 1e-4
