"""-m gpu: Philox4x32-10 of both sides against cuRAND's own Philox4_32_10 (SURVEY.md 8(c) "Pins", Philox row: "on the GPU
box also cross-check against cuRAND's Philox4_32_10 raw output").

cuRAND's device API fixes the generator's layout: curand_init(seed, subsequence, offset, &state) sets key = (seed lo,
seed hi) and counter = (offset / 4 as 64 bits in words 0-1, subsequence as 64 bits in words 2-3); curand4() returns the
four output words of that counter and increments it.  With subsequence = slot | component << 32 and offset = 4 i this is
the (i lo, i hi, slot, component) counter of DESIGN.md section 2 step 1.  The helper below (a test program, compiled here
with nvcc from cuRAND's public header, not part of the product) dumps raw words; the oracle's orc_philox must equal them,
and so must the words behind the product's draws (checked through mcx_trace_dump on a source whose bin index is the
draw).
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SRC = r'''
#include <curand_kernel.h>
#include <stdint.h>
__global__ void dump(uint64_t seed, const uint64_t* sub, const uint64_t* idx, int n, uint32_t* out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  curandStatePhilox4_32_10_t st;
  curand_init(seed, sub[k], 4ull * idx[k], &st);
  const uint4 w = curand4(&st);
  out[4 * k + 0] = w.x; out[4 * k + 1] = w.y; out[4 * k + 2] = w.z; out[4 * k + 3] = w.w;
}
extern "C" int curand_philox_raw(uint64_t seed, const uint64_t* sub_h, const uint64_t* idx_h, int n, uint32_t* out_h) {
  uint64_t *sub, *idx; uint32_t* out;
  if (cudaMalloc(&sub, 8 * n) || cudaMalloc(&idx, 8 * n) || cudaMalloc(&out, 16 * n)) return 1;
  cudaMemcpy(sub, sub_h, 8 * n, cudaMemcpyHostToDevice);
  cudaMemcpy(idx, idx_h, 8 * n, cudaMemcpyHostToDevice);
  dump<<<(n + 127) / 128, 128>>>(seed, sub, idx, n, out);
  const int rc = cudaMemcpy(out_h, out, 16 * n, cudaMemcpyDeviceToHost) != cudaSuccess;
  cudaFree(sub); cudaFree(idx); cudaFree(out);
  return rc ? 2 : 0;
}
'''


@pytest.fixture(scope="module")
def curand(tmp_path_factory):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    d = tmp_path_factory.mktemp("curand")
    src, lib = os.path.join(d, "curand_philox.cu"), os.path.join(d, "libcurand_philox.so")
    open(src, "w").write(SRC)
    nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-shared", "-Xcompiler", "-fPIC", "-o", lib, src])
    L = C.CDLL(lib)
    L.curand_philox_raw.argtypes = [C.c_uint64, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]

    def raw(seed, sub, idx):
        sub, idx = np.ascontiguousarray(sub, dtype=np.uint64), np.ascontiguousarray(idx, dtype=np.uint64)
        out = np.zeros((len(sub), 4), dtype=np.uint32)
        assert L.curand_philox_raw(seed, sub.ctypes.data, idx.ctypes.data, len(sub), out.ctypes.data) == 0
        return out
    return raw


def test_oracle_philox_equals_curand_raw_output(curand, O):
    rng = np.random.default_rng(3)
    for seed in (0, 1, 0xDEADBEEFCAFEF00D, 2**64 - 1):
        idx = np.concatenate([[0, 1, 2, 2**32 - 1, 2**32, 2**40 + 7], rng.integers(0, 2**62, size=200, dtype=np.uint64)]).astype(np.uint64)
        slot = rng.integers(0, 8, size=len(idx)).astype(np.uint64)
        comp = rng.integers(0, 16, size=len(idx)).astype(np.uint64)
        words = curand(seed, slot | (comp << np.uint64(32)), idx)
        for k in range(len(idx)):
            i = int(idx[k])
            mine = O.philox((i & 0xFFFFFFFF, i >> 32, int(slot[k]), int(comp[k])), (seed & 0xFFFFFFFF, seed >> 32))
            assert mine == tuple(int(x) for x in words[k]), (seed, i)


def test_product_draws_equal_curand_raw_output(curand, W):
    """The product exports no raw Philox call; its slot-1 draw of the source decides where a ray of a point source lands
    on a fine detector (u = (top 52 bits of (w0:w1) + 1/2) 2^-52, x = (u - 1/2) w).  With a 2^10 x 2^10 detector over
    the target the bin index of ray i IS the top 10 bits of w0 and of w2 of cuRAND's output for (seed, i, slot 1)."""
    import torch  # noqa: F401
    import paper_2410_08747_b200 as M
    src = W.source("point", "target", "mono", target_w=0.1024, target_h=0.1024, target_dist=1.0, E0=20.0)
    det = W.detector(-0.0512, 0.0512, -0.0512, 0.0512, 1024, 1024, 0.0, 40.0, 1, T=(0, 0, 1.0))
    inst = W.instrument("philox_bits", [src, det], [None], 1000)
    for seed, first in ((1, 0), (0x0123456789ABCDEF, 2**33 + 5)):
        g = M.Instrument(inst)
        d = g.trace_dump(first, 20_000, seed)
        g.close()
        idx = np.arange(first, first + 20_000, dtype=np.uint64)
        words = curand(seed, np.full(len(idx), 1, dtype=np.uint64), idx)          # slot 1, component 0
        ix, iy = words[:, 0] >> 22, words[:, 2] >> 22
        expect = iy.astype(np.int64) * 1024 + ix.astype(np.int64)
        # a ray within 1e-13 of a pixel edge may round across it on its way through the plane intersection
        assert (d["bin"] != expect).sum() <= 2
        assert np.all(d["fate"] == M.binding.FATE_DETECTED)
