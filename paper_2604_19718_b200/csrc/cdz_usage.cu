// cdz_usage.cu -- finishing kernels of the outside pass (sm_100a): from the adjoint tables to the operator usages
//   u_z = x_z dlogZ/dx_z = P(operator z is used at its position),
// and from them the base marginals (eq 2.6 line 90 / eq 4.2), the codon marginals (eq 2.7 line 96 / eq 4.3) and
// the unpaired probabilities.  Roles an operator can play (cdz_outside.h): pair end (left / right), closing / inner mismatch of a loop,
// size-1 bulge, interior of an unpaired stretch E (hairpin interiors and loop sides), unpaired in a multiloop (leading, via Qml; trailing,
// via Qm1), unpaired in the exterior loop.  The roles are disjoint events and every position uses exactly one operator, so
// sum_z u_z = 1 at every position -- checked on the device (status flag), never enforced.
#include <math.h>

#include "cdz_outside.h"

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_dot(const double* __restrict__ x, const double* __restrict__ y, int k0, int k1, int lane) {
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  int k = k0 + lane;
  for (; k + 96 < k1; k += 128) {
    a0 += x[k] * y[k];
    a1 += x[k + 32] * y[k + 32];
    a2 += x[k + 64] * y[k + 64];
    a3 += x[k + 96] * y[k + 96];
  }
  for (; k < k1; k += 32) a0 += x[k] * y[k];
  return warp_sum((a0 + a1) + (a2 + a3));
}

// E-bar chain: E(s,e) = E(s,e-1) Tbar_e, so  E-bar(s,e-1) += E-bar(s,e) Tbar_e^T.  One thread per bond row (s,a) walks e = n-1 .. s; the seeds
// are the hairpin interiors already in AET and the loop-side stretches of the per-role accumulators.  AET is transposed (row (e+1,c),
// column (s,a)), so the threads of a warp read consecutive addresses.
__global__ void __launch_bounds__(128) echain_kernel(const Ctx* ctx, Adj A) {
  const DevTT& t = ctx->tt;
  const int n = t.n, MS = t.MS, MS2 = MS * MS;
  const size_t S = (size_t)t.S;
  const int R = blockIdx.x * blockDim.x + threadIdx.x;
  if (R >= t.S) return;
  const int s = t.bondpos[R];
  if (s >= n) return;
  const int a = R - t.off[s];
  if (a < 0 || a >= t.sig[s]) return;  // padding row of the block
  double carry[CDZ_MAX_BOND];
#pragma unroll
  for (int c = 0; c < CDZ_MAX_BOND; ++c) carry[c] = 0.0;
  for (int e = n - 1; e >= s; --e) {
    const int Se1 = t.sig[e + 1], Se = t.sig[e], len = e - s + 1;
    double v[CDZ_MAX_BOND];
#pragma unroll
    for (int c = 0; c < CDZ_MAX_BOND; ++c) {
      v[c] = 0.0;
      if (c < Se1) {
        double x = A.AET[(size_t)(t.off[e + 1] + c) * S + R] + carry[c];
        if (len < SLEN)
          for (int role = 0; role < AES_NROLE; ++role) x += A.AES[(((size_t)role * n + s) * SLEN + len) * MS2 + a * MS + c];
        A.AET[(size_t)(t.off[e + 1] + c) * S + R] = x;
        v[c] = x;
      }
    }
    const double* Tb = t.Tbar + (size_t)e * MS2;
#pragma unroll
    for (int c2 = 0; c2 < CDZ_MAX_BOND; ++c2) {
      double w = 0.0;
      if (c2 < Se)
#pragma unroll
        for (int c = 0; c < CDZ_MAX_BOND; ++c)
          if (c < Se1) w += v[c] * Tb[c2 * MS + c];
      carry[c2] = w;
    }
  }
}

// One CTA per position m: the four table-row usages of every operator at m, the totals over roles, the marginals and the checks.
__global__ void __launch_bounds__(256) usage_kernel(const Ctx* ctx, Adj A, double* __restrict__ bpp, double* __restrict__ base,
                                                    double* __restrict__ codon) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const CModel& cm = *ctx->cm;
  const int n = t.n, MS = t.MS;
  const size_t S = (size_t)t.S, no = A.nops;
  const int m = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int z0 = t.opstart[m], nz = t.opstart[m + 1] - z0;
  const int send = t.off[n] + t.sig[n];
  __shared__ double tot[64], pairu[64];
  for (int k = warp; k < nz; k += 8) {
    const int z = z0 + k, a = t.op_a[z], c = t.op_c[z];
    const double x = t.op_x[z];
    // interior of an unpaired stretch: sum_{(s,a') : s <= m} E(s,m-1)[a',a] E-bar(s,m)[a',c]
    const double ue = warp_dot(b.EMT + (size_t)(t.off[m] + a) * S, A.AET + (size_t)(t.off[m + 1] + c) * S, 0, t.off[m] + t.sig[m], lane);
    // unpaired, leading a multiloop segment: Qml(m,j) = .. + w_b T_m Qml(m+1,j)
    double uml = 0.0, um1 = 0.0;
    if (m + 1 <= n - 1)
      uml = warp_dot(A.AML + (size_t)(t.off[m] + a) * S, b.QML + (size_t)(t.off[m + 1] + c) * S, t.off[m + 2], send, lane);
    // unpaired, trailing a multiloop branch: Qm1(i,m) = .. + w_b Qm1(i,m-1) T_m
    if (m >= 1) um1 = warp_dot(A.AM1T + (size_t)(t.off[m + 1] + c) * S, b.QM1T + (size_t)(t.off[m] + a) * S, 0, t.off[m], lane);
    if (lane == 0) {
      A.U[(size_t)ROLE_E * no + z] = x * ue;
      A.U[(size_t)ROLE_ML * no + z] = cm.wb * x * uml;
      A.U[(size_t)ROLE_M1 * no + z] = cm.wb * x * um1;
      // unpaired in the exterior loop: Qext(m) = Qext(m-1) T_m + ..
      A.U[(size_t)ROLE_EXT * no + z] = b.Qext[t.off[m] + a] * x * A.AX[(size_t)(m + 1) * MS + c];
    }
  }
  __syncthreads();
  if (tid < nz) {
    double s = 0.0;
    for (int role = 0; role < NROLE; ++role) s += A.U[(size_t)role * no + z0 + tid];
    tot[tid] = s;
    pairu[tid] = A.U[(size_t)ROLE_PL * no + z0 + tid] + A.U[(size_t)ROLE_PR * no + z0 + tid];
  }
  __syncthreads();
  if (tid == 0) {
    double all = 0.0, paired = 0.0, bs[4] = {0.0, 0.0, 0.0, 0.0};
    bool bad = false;
    for (int k = 0; k < nz; ++k) {
      all += tot[k];
      paired += pairu[k];
      bs[t.op_b[z0 + k]] += tot[k];
      if (!(tot[k] >= -1e-9 && tot[k] <= 1.0 + 1e-9)) bad = true;
      if (codon && t.op_codon[z0 + k] >= 0) codon[(size_t)(m / 3) * 64 + t.op_codon[z0 + k]] = tot[k];
    }
    if (!(fabs(all - 1.0) <= 1e-6)) bad = true;  // also catches NaN / inf
    if (base)
      for (int x = 0; x < 4; ++x) base[(size_t)m * 4 + x] = bs[x];
    if (bpp) bpp[(size_t)m * n + m] = all - paired;  // P(m unpaired): from the unpaired roles, independent of the pair sums
    if (bad) atomicOr(A.status, 1);
  }
}

}  // namespace

int cdz_launch_usage(cdz_tables* t, const Adj& A, double* bpp_dev, double* base_dev, double* codon_dev, cudaStream_t st) {
  const cdz_tt* tt = t->tt;
  const int n = tt->n;
  if (codon_dev) CDZ_CUDA(cudaMemsetAsync(codon_dev, 0, sizeof(double) * (size_t)(n / 3) * 64, st));
  echain_kernel<<<(tt->S + 127) / 128, 128, 0, st>>>(t->d_ctx, A);
  usage_kernel<<<n, 256, 0, st>>>(t->d_ctx, A, bpp_dev, base_dev, codon_dev);
  CDZ_CUDA(cudaGetLastError());
  return CDZ_OK;
}
