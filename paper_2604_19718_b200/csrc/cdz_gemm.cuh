// cdz_gemm.cuh -- the fp64 tensor-core tile product shared by the split-point GEMM of the inside pass (cdz_inside.cu, gemm_kernel) and the
// TRMM-with-dependency of the tensor-model recursion (cdz_tm.cu, tm_gemm_kernel):
//     C[64 x 64] = A[64 rows, kbeg..kend) * Bm[64 rows, kbeg..kend)^T
// Both operands are K-contiguous row-major panels with row stride S (the paper's flattened product Q_{i,k} Q_{j,k}^T, eq 3.5,
// TRMM of eq S4.1).  fp64 mma.sync m8n8k4 (DMMA; tcgen05.mma has no f64 kind), 3-stage cp.async pipeline, 128 threads, each warp a
// 32 x 32 sub-tile.  kbeg, kend are multiples of GEMM_BK.
#pragma once
#include <cuda_runtime.h>

#include "cdz_internal.h"

constexpr int GEMM_BK = 16, GEMM_LD = 20, GEMM_STAGES = 3, GEMM_THREADS = 128;
constexpr int GEMM_SMEM = GEMM_STAGES * 2 * CDZ_TB * GEMM_LD * (int)sizeof(double);

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem_src));
}
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

// gsm: GEMM_SMEM bytes of dynamic shared memory; C: 64 x 64 row-major output tile (row stride CDZ_TB)
__device__ __forceinline__ void cdz_gemm_tile(const double* __restrict__ A, const double* __restrict__ Bm, size_t S, int kbeg, int kend,
                                              double* __restrict__ C, double* gsm) {
  double* As = gsm;
  double* Bs = gsm + GEMM_STAGES * CDZ_TB * GEMM_LD;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;

  auto load_stage = [&](int st, int kk) {
    double* as = As + st * CDZ_TB * GEMM_LD;
    double* bs = Bs + st * CDZ_TB * GEMM_LD;
#pragma unroll
    for (int r = 0; r < (CDZ_TB * GEMM_BK / 2) / GEMM_THREADS; ++r) {
      const int c = tid + r * GEMM_THREADS, row = c >> 3, ch = (c & 7) * 2;
      cp_async16(as + row * GEMM_LD + ch, A + (size_t)row * S + kk + ch);
      cp_async16(bs + row * GEMM_LD + ch, Bm + (size_t)row * S + kk + ch);
    }
  };

  double acc[4][4][2];
#pragma unroll
  for (int mi = 0; mi < 4; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;

  const int nkt = (kend - kbeg) / GEMM_BK;
#pragma unroll
  for (int st = 0; st < GEMM_STAGES - 1; ++st) {
    if (st < nkt) load_stage(st, kbeg + st * GEMM_BK);
    asm volatile("cp.async.commit_group;\n" ::);
  }
  for (int kt = 0; kt < nkt; ++kt) {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(GEMM_STAGES - 2));
    __syncthreads();
    const int nxt = kt + GEMM_STAGES - 1;
    if (nxt < nkt) load_stage(nxt % GEMM_STAGES, kbeg + nxt * GEMM_BK);
    asm volatile("cp.async.commit_group;\n" ::);
    const double* as = As + (kt % GEMM_STAGES) * CDZ_TB * GEMM_LD + (wm + (lane >> 2)) * GEMM_LD + (lane & 3);
    const double* bs = Bs + (kt % GEMM_STAGES) * CDZ_TB * GEMM_LD + (wn + (lane >> 2)) * GEMM_LD + (lane & 3);
#pragma unroll
    for (int k4 = 0; k4 < GEMM_BK / 4; ++k4) {
      double af[4], bf[4];
#pragma unroll
      for (int mi = 0; mi < 4; ++mi) af[mi] = as[mi * 8 * GEMM_LD + k4 * 4];
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) bf[ni] = bs[ni * 8 * GEMM_LD + k4 * 4];
#pragma unroll
      for (int mi = 0; mi < 4; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) dmma884(acc[mi][ni], af[mi], bf[ni]);
    }
  }
  asm volatile("cp.async.wait_group 0;\n" ::);
#pragma unroll
  for (int mi = 0; mi < 4; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) {
      const int r = wm + mi * 8 + (lane >> 2), c = wn + ni * 8 + 2 * (lane & 3);
      *reinterpret_cast<double2*>(C + r * CDZ_TB + c) = make_double2(acc[mi][ni][0], acc[mi][ni][1]);
    }
}
