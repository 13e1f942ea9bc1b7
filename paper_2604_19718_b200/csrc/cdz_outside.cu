// cdz_outside.cu -- outside (adjoint) pass over the stored inside tables (sm_100a): base-pair probabilities (eq 2.5 line 85,
// eq 4.1) and the operator usages  u_z = x_z dlogZ/dx_z  from which the base marginals (eq 2.6 line 90, eq 4.2) and the
// codon marginals (eq 2.7 line 96, eq 4.3) follow (the paper's ComputeReverse, Alg S4.3, re-expressed
// as the reverse-mode adjoint of the recursion of DESIGN.md section 3).
//
// All adjoints are derivatives of log Z with respect to the STORED (scaled) table entries; a power-of-two scale per position is a change of
// operator weights under which the recursion is unchanged, so every probability  entry x adjoint  is scale-free.
//
// Diagonals d = n-1 .. 0, one launch each, one CTA per cell (i, j = i+d).  Per cell, in this order:
//   1  bond-level adjoints (the two split-point gathers are dot products of contiguous table rows: QM1 / QMT are plain transposes made
//      at the start of the call, AM2T is written beside AM2):
//        Qm-bar(i,j)  = sum_{j'>j} M2-bar(i,j') Qm1(j+1,j')^T            M2-bar = Qm-bar + w_a w_c sum_{x,y} I(i-1,j+1)[x,y]
//        Qml-bar      = Qm-bar + w_b Tbar_{i-1}^T Qml-bar(i-1,j)
//        Qm1-bar      = Qml-bar + w_b Qm1-bar(i,j+1) Tbar_{j+1}^T + sum_{i'<i} Qm(i',i-1)^T M2-bar(i',j)
//        Qbs-bar      = w_c Qm1-bar + Qext(i-1)^T Qext-bar(j+1)
//   2  Qb-bar(i,j) = Qbs-bar + stack / bulge terms pulled from the I tables of the <= 61 closing pairs (ring of 36 diagonals)
//                  + the interior-loop terms, which closing cells PUSHED earlier into this cell's ring slot as adjoints of its dressed
//                    extensions DD / D1 / D2T / GI;   P(i.j) = sum Qb (.) Qb-bar;   usages of the inner-mismatch operators at i-1, j+1
//   3  I = adjoint of `inner`, G = I with the closing mismatch applied, H / H1 / H2 = G with the loop-side operators contracted
//      (= adjoints of the loop bodies XE, Z1, Z2 of the inside pass)
//   4  as closing pair: adjoint row / column recursions of the interior-loop bodies X_u (27 small products per cell instead of 378),
//      pushes into the ring slots of the inner cells and into the stretch adjoints E-bar (hairpin interiors: table AET; loop sides:
//      per-role accumulators AES), and -- with `inner`, Y, Z1, Z2, Bl, Br, SB recomputed from the stored tables exactly as the inside
//      pass does -- the usages of the operators at i, j (pair ends), i+1, j-1 (closing mismatch, size-1 bulges).
// Every accumulator has a single writer per launch (role-separated), every sum a fixed order: results are bit-reproducible.
// cdz_usage.cu finishes: E-bar chain, multiloop / exterior unpaired usages, base / codon marginals, unpaired probabilities.
#include <vector>

#include "cdz_outside.h"

#ifdef CDZ_OTIMING
#include <stdio.h>
__device__ unsigned long long g_otime[16], g_omax[16];
#define OTICK(k) do { __syncthreads(); if (threadIdx.x == 0) { const long long now__ = clock64(); atomicAdd(&g_otime[k], (unsigned long long)(now__ - tlast__)); atomicMax(&g_omax[k], (unsigned long long)(now__ - tlast__)); tlast__ = now__; } } while (0)
#else
#define OTICK(k)
#endif

namespace {

constexpr int OT = 256;  // threads per CTA (512 measured slower: 0.33 vs 0.30 s at config 2)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// All nx x ny dot products  out[a * ny + c] = sum_{kb in [k0,k1)} X[a * S + kb] Y[c * S + kb]  of two small groups of table rows at once: every
// thread strides the bond range (coalesced), loads the nx + ny values of its column once and keeps the nx x ny accumulators; warp shuffle
// trees, then a fixed-order sum over the warps.  MSX = compile-time bound of nx, ny (4 or 8).
template <int MSX, int NT_>
__device__ __forceinline__ void gather_all(const double* __restrict__ X, int nx, const double* __restrict__ Y, int ny, size_t S, int k0,
                                           int k1, double* out, double* red) {
  constexpr int RC = MSX == 4 ? 4 : 2;  // rows per pass: 16 accumulators per thread (register budget of 4 CTAs per SM)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int a0 = 0; a0 < nx; a0 += RC) {
    double acc[RC][MSX];
#pragma unroll
    for (int a = 0; a < RC; ++a)
#pragma unroll
      for (int c = 0; c < MSX; ++c) acc[a][c] = 0.0;
    for (int kb = k0 + (int)threadIdx.x; kb < k1; kb += NT_) {
      double x[RC], y[MSX];
#pragma unroll
      for (int a = 0; a < RC; ++a) x[a] = a0 + a < nx ? X[(size_t)(a0 + a) * S + kb] : 0.0;
#pragma unroll
      for (int c = 0; c < MSX; ++c) y[c] = c < ny ? Y[(size_t)c * S + kb] : 0.0;
#pragma unroll
      for (int a = 0; a < RC; ++a)
#pragma unroll
        for (int c = 0; c < MSX; ++c) acc[a][c] += x[a] * y[c];
    }
#pragma unroll
    for (int a = 0; a < RC; ++a)
#pragma unroll
      for (int c = 0; c < MSX; ++c) {
        if (a0 + a < nx && c < ny) {  // (uniform across the CTA)
          const double v = warp_sum(acc[a][c]);
          if (lane == 0) red[warp * (MSX * MSX) + (a0 + a) * MSX + c] = v;
        }
      }
  }
  __syncthreads();
  if ((int)threadIdx.x < nx * ny) {
    const int a = threadIdx.x / ny, c = threadIdx.x % ny;
    double v = 0.0;
    for (int w = 0; w < NT_ / 32; ++w) v += red[w * (MSX * MSX) + a * MSX + c];
    out[a * ny + c] = v;
  }
  __syncthreads();
}

// Qext-bar, sequential over bond positions k = n .. 0 (one CTA):  AX(k) = Tbar_k AX(k+1) + sum_{j>=k} Qbs(k,j) AX(j+1), AX(n) = 1/Z
__global__ void __launch_bounds__(1024) oext_kernel(const Ctx* ctx, Adj A) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const int n = t.n, S = t.S, MS = t.MS;
  __shared__ double part[32][CDZ_MAX_BOND];
  __shared__ double zinv;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  if (tid == 0) {
    double Z = 0.0;
    for (int c = 0; c < t.sig[n]; ++c) Z += b.Qext[t.off[n] + c];
    zinv = 1.0 / Z;
  }
  __syncthreads();
  // AXB: Qext-bar laid out over the bond index space (AXB[off[k]+s]) so that the gather is a dot product with a row of QBS
  for (int k = tid; k < S; k += blockDim.x) A.AXB[k] = 0.0;
  __syncthreads();
  if (tid < t.sig[n]) { A.AX[(size_t)n * MS + tid] = zinv; A.AXB[t.off[n] + tid] = zinv; }
  __syncthreads();
  const int send = t.off[n] + t.sig[n];
  for (int k = n - 1; k >= 0; --k) {
    const int Sk = t.sig[k], ok = t.off[k], k0 = t.off[k + 1];
    // every warp takes a slice of the bond range [off[k+1], send) for all s < Sk
    const int len = send - k0, per = (len + nwarp - 1) / nwarp;
    const int w0 = k0 + warp * per, w1 = min(send, w0 + per);
    for (int s = 0; s < Sk; ++s) {
      const double* q = b.QBS + (size_t)(ok + s) * S;
      double acc = 0.0;
      for (int kb = w0 + lane; kb < w1; kb += 32) acc += q[kb] * A.AXB[kb];
      acc = warp_sum(acc);
      if (lane == 0) part[warp][s] = acc;
    }
    __syncthreads();
    if (tid < Sk) {
      double v = 0.0;
      for (int w = 0; w < nwarp; ++w) v += part[w][tid];
      for (int c = 0; c < t.sig[k + 1]; ++c) v += t.Tbar[((size_t)k * MS + tid) * MS + c] * A.AX[(size_t)(k + 1) * MS + c];
      A.AX[(size_t)k * MS + tid] = v;
      A.AXB[ok + tid] = v;
    }
    __syncthreads();
  }
}

// plain copies with the other orientation, upper block triangle only: QM1[(j+1,s)][(j'+1,c)] from QM1T, QMT[(k,s)][(i,a)] from QM
__global__ void __launch_bounds__(256) transpose_kernel(const double* __restrict__ src, double* __restrict__ dst, int S, int src_lower) {
  __shared__ double tile[CDZ_TB][CDZ_TB + 1];
  const int bi = blockIdx.y, bj = blockIdx.x;  // source tile (bi, bj)
  if (src_lower ? (bj > bi) : (bj < bi)) return;
  for (int e = threadIdx.x; e < CDZ_TB * CDZ_TB; e += blockDim.x) {
    const int r = e / CDZ_TB, c = e % CDZ_TB;
    tile[r][c] = src[(size_t)(bi * CDZ_TB + r) * S + bj * CDZ_TB + c];
  }
  __syncthreads();
  for (int e = threadIdx.x; e < CDZ_TB * CDZ_TB; e += blockDim.x) {
    const int r = e / CDZ_TB, c = e % CDZ_TB;
    dst[(size_t)(bj * CDZ_TB + r) * S + bi * CDZ_TB + c] = tile[c][r];
  }
}

// shared-memory plan of ocell_kernel (doubles); identical on host and device
struct OPlan {
  int am, aml, abs_, ab, qb, ibs, go, h, h1, h2, ibsum, sbb, xe, bl, br, z1, z2, sb, y, inn, ddb, tl, tr, part, red, total;
};
__host__ __device__ inline OPlan oplan(int MS, int ML, int MR, int nps) {
  OPlan p;
  const int MS2 = MS * MS;
  int o = 0;
  auto take = [&](int k) { int r = o; o += (k + 1) & ~1; return r; };
  p.am = take(MS2); p.aml = take(MS2); p.abs_ = take(MS2);
  p.ab = take(ML * MR); p.qb = take(ML * MR);
  p.ibs = take(nps * MS2); p.go = take(16 * MS2);
  p.h = take(MS2); p.h1 = take(4 * MS2); p.h2 = take(4 * MS2);
  p.ibsum = take(MS2); p.sbb = take(nps * MS2);
  p.xe = take(MS2); p.bl = take(MS2); p.br = take(MS2);
  p.z1 = take(ML * MS); p.z2 = take(MS * MR);
  p.sb = take(nps * MS2); p.y = take(ML * MR > 4 * MS * MR ? ML * MR : 4 * MS * MR); p.inn = take(nps * MS2);
  p.ddb = take(ML * MR);
  p.tl = take(3 * ML * MS); p.tr = take(3 * MS * MR);
  p.part = take(OT);
  p.red = take((OT / 32) * 64);
  p.total = o;
  return p;
}

// deterministic block sum of per-thread partials laid out as [group][entry]: entry e = tid % nent, group tid / nent
__device__ __forceinline__ double group_total(double* part, double v, int nent) {
  __syncthreads();
  part[threadIdx.x] = v;
  __syncthreads();
  double s = 0.0;
  if ((int)threadIdx.x < nent)
    for (int g = 0; g < OT / nent; ++g) s += part[g * nent + threadIdx.x];
  return s;
}

// PART 0: phases 1-3 and 4a-4b, the chain every later diagonal waits for; leaves Qb-bar, the pushed adjoints it consumed, G, H1, H2, sum I
// and SB-bar of the cell in a scratch record.  PART 1: everything that only later consumers need (the pushes into the inner cells at least
// four diagonals below, the stretch adjoints, the usages), run on a second stream so that it overlaps the chain of the next diagonals.
template <int PART, int MSX>
__global__ void __launch_bounds__(OT, 4) ocell_kernel(const Ctx* ctx, Adj A, int d, int want_usage, double* __restrict__ bpp) {
  extern __shared__ double osm[];
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const CModel& m = *ctx->cm;
  const int n = t.n, MS = t.MS, MS2 = MS * MS, tid = threadIdx.x;
  const size_t S = (size_t)t.S, RS = (size_t)t.RS;
  const int ML = A.ML, MR = A.MR, nps = m.nps;
  const OPlan pl = oplan(MS, ML, MR, nps);
  double *am = osm + pl.am, *aml = osm + pl.aml, *abs_ = osm + pl.abs_, *ab = osm + pl.ab, *qbv = osm + pl.qb, *ibs = osm + pl.ibs,
         *go = osm + pl.go, *h = osm + pl.h, *h1 = osm + pl.h1, *h2 = osm + pl.h2, *ibsum = osm + pl.ibsum, *sbb = osm + pl.sbb,
         *xe = osm + pl.xe, *bl = osm + pl.bl, *br = osm + pl.br, *z1 = osm + pl.z1, *z2 = osm + pl.z2, *sb = osm + pl.sb,
         *y = osm + pl.y, *inn = osm + pl.inn, *ddb = osm + pl.ddb, *part = osm + pl.part, *red = osm + pl.red;
  double* TLm = osm + pl.tl;            // T_{i-1}[lst][c]   (ML x MS)
  double* TLi = TLm + ML * MS;          // T_i
  double* TLp = TLi + ML * MS;          // T_{i+1}
  double* TRq = osm + pl.tr;            // T_{j-1}[a][r]     (MS x MR)
  double* TRj = TRq + MS * MR;          // T_j
  double* TRn = TRj + MS * MR;          // T_{j+1}

#ifdef CDZ_OTIMING
  long long tlast__ = clock64();
#endif
  const int i = blockIdx.x, j = i + d, p = i + 1, q = j - 1;
  const int Si = t.sig[i], Sj1 = t.sig[j + 1], offi = t.off[i], offj1 = t.off[j + 1];
  const int nent = Si * Sj1;
  const int mh1 = m.min_hairpin + 1, MI = m.max_interior;
  const bool closed = d >= mh1;
  const int nL = t.loff[i + 1] - t.loff[i], nR = t.roff[j + 1] - t.roff[j], npair = nL * nR;
  const int Li0 = t.loff[i], Rj0 = t.roff[j];
  const int send = t.off[n] + t.sig[n];

  // ---- offsets / bond dimensions of the positions within 35 of i and of j (loop sides reach 31 positions) ----------------------------------
  __shared__ int offW[2][72], sigW[2][72];
  if (tid < 144) {
    const int which = tid / 72, idx = tid % 72, pos = (which ? j : i) - 35 + idx;
    const bool ok = pos >= 0 && pos <= n;
    offW[which][idx] = ok ? t.off[pos] : 0;
    sigW[which][idx] = ok ? t.sig[pos] : 0;
  }
  // boundary states of positions i-1, i, i+1 (left states) and j-1, j, j+1 (right states)
  __shared__ uint8_t sLa[3][CDZ_MAX_STATES], sLx[3][CDZ_MAX_STATES], sRy[3][CDZ_MAX_STATES], sRc[3][CDZ_MAX_STATES];
  if (tid >= 160 && tid < 160 + 6 * CDZ_MAX_STATES) {
    const int w6 = (tid - 160) / CDZ_MAX_STATES, k = (tid - 160) % CDZ_MAX_STATES;
    const int pos = w6 < 3 ? i - 1 + w6 : j - 1 + (w6 - 3);
    if (pos >= 0 && pos < n) {
      if (w6 < 3) {
        const int l0 = t.loff[pos], nl = t.loff[pos + 1] - l0;
        if (k < nl) { sLa[w6][k] = t.ls_a[l0 + k]; sLx[w6][k] = t.ls_x[l0 + k]; }
      } else {
        const int r0 = t.roff[pos], nr = t.roff[pos + 1] - r0;
        if (k < nr) { sRy[w6 - 3][k] = t.rs_y[r0 + k]; sRc[w6 - 3][k] = t.rs_c[r0 + k]; }
      }
    }
  }
  auto offA = [&](int pos) { return offW[0][pos - i + 35]; };
  auto sigA = [&](int pos) { return sigW[0][pos - i + 35]; };
  auto offB = [&](int pos) { return offW[1][pos - j + 35]; };
  auto sigB = [&](int pos) { return sigW[1][pos - j + 35]; };
  // E(p,q)[a][c] with p and q+1 near i (EA) / near j (EB)
  auto EA = [&](int pp, int qq, int a, int c) { return qq < pp ? (a == c ? 1.0 : 0.0) : b.EM[(size_t)(offA(pp) + a) * S + offA(qq + 1) + c]; };
  auto EB = [&](int pp, int qq, int a, int c) { return qq < pp ? (a == c ? 1.0 : 0.0) : b.EM[(size_t)(offB(pp) + a) * S + offB(qq + 1) + c]; };
  // ---- dense cores of the six positions around the cell ------------------------------------------------------------------------------
  for (int k = tid; k < 3 * ML * MS + 3 * MS * MR; k += OT) (k < 3 * ML * MS ? TLm[k] : TRq[k - 3 * ML * MS]) = 0.0;
  __syncthreads();
  {
    // one thread per operator of the six positions (<= 36 each); distinct operators hit distinct core entries, duplicates of a generic
    // operator list add up (shared-memory atomics)
    for (int e = tid; e < 6 * 64; e += OT) {
      const int w6 = e / 64, k = e % 64;
      const int pos = w6 < 3 ? i - 1 + w6 : j - 1 + (w6 - 3);
      if (pos < 0 || pos >= n) continue;
      const int z0 = t.opstart[pos], nz = t.opstart[pos + 1] - z0;
      for (int zz = k; zz < nz; zz += 64) {
        const int z = z0 + zz;
        if (w6 < 3) atomicAdd(&TLm[w6 * ML * MS + t.op_l[z] * MS + t.op_c[z]], t.op_x[z]);
        else atomicAdd(&TRq[(w6 - 3) * MS * MR + t.op_a[z] * MR + t.op_r[z]], t.op_x[z]);
      }
    }
  }
  if constexpr (PART == 0) {
  // ---- 1: bond-level adjoints ------------------------------------------------------------------------------------------------------------
  // Qm-bar(i,j)[a,s] = sum_{kb >= off[j+2]} AM2[(i,a)][kb] QM1[(j+1,s)][kb]
  if (j + 1 <= n - 1) {
    gather_all<MSX, OT>(A.AM2 + (size_t)offi * S, Si, A.QM1 + (size_t)offj1 * S, Sj1, S, t.off[j + 2], send, am, red);
  } else {
    if (tid < nent) am[tid] = 0.0;
    __syncthreads();
  }
  if (tid < nent) {
    const int ea = tid / Sj1, ec = tid % Sj1;
    // M2-bar = Qm-bar + w_a w_c sum_{x,y} I(i-1,j+1)[x,y]
    double v = am[tid];
    if (i >= 1 && j + 1 <= n - 1) {
      const double* ib = A.IB + ((size_t)((d + 2) % ORING) * n + (i - 1)) * 16 * MS2 + ea * MS + ec;
      double s = 0.0;
      for (int sl = 0; sl < nps; ++sl) s += ib[sl * MS2];
      v += m.wac * s;
    }
    A.AM2[(size_t)(offi + ea) * S + offj1 + ec] = v;
    A.AM2T[(size_t)(offj1 + ec) * S + offi + ea] = v;
    // Qml-bar = Qm-bar + w_b Tbar_{i-1}^T Qml-bar(i-1,j)
    double w = am[tid];
    if (i >= 1) {
      double s = 0.0;
      for (int a = 0; a < t.sig[i - 1]; ++a)
        s += t.Tbar[((size_t)(i - 1) * MS + a) * MS + ea] * A.AML[(size_t)(t.off[i - 1] + a) * S + offj1 + ec];
      w += m.wb * s;
    }
    aml[tid] = w;
    A.AML[(size_t)(offi + ea) * S + offj1 + ec] = w;
  }
  // Qm1-bar = Qml-bar + w_b Qm1-bar(i,j+1) Tbar_{j+1}^T + sum_{rb < off[i]} QMT[(i,a)][rb] AM2T[(j+1,c)][rb]
  gather_all<MSX, OT>(A.QMT + (size_t)offi * S, Si, A.AM2T + (size_t)offj1 * S, Sj1, S, 0, offi, abs_, red);
  if (tid < nent) {
    const int ea = tid / Sj1, ec = tid % Sj1;
    double w = aml[tid] + abs_[tid];
    if (j + 1 <= n - 1) {
      double s = 0.0;
      for (int c2 = 0; c2 < t.sig[j + 2]; ++c2)
        s += A.AM1T[(size_t)(t.off[j + 2] + c2) * S + offi + ea] * t.Tbar[((size_t)(j + 1) * MS + ec) * MS + c2];
      w += m.wb * s;
    }
    A.AM1T[(size_t)(offj1 + ec) * S + offi + ea] = w;
    // Qbs-bar = w_c Qm1-bar + Qext(i-1)^T Qext-bar(j+1)
    abs_[tid] = m.wc * w + b.Qext[offi + ea] * A.AX[(size_t)(j + 1) * MS + ec];
  }
  __syncthreads();
  }
  OTICK(0);
  if (!closed) {
    if constexpr (PART == 1) return;
    // cells below the minimum hairpin span: nothing pairs and none of their loop bodies exists
    if (d >= 4) {
      double* xa = A.XA + ((size_t)(d % XRING) * n + i) * XU * MS2;
      double* xb = A.XB + ((size_t)(d % XRING) * n + i) * XU * MS2;
      for (int e = tid; e < XU * MS2; e += OT) { xa[e] = 0.0; xb[e] = 0.0; }
    }
    // the I slot of this diagonal is read by the M2-bar of cell (i+1, j-1): it must not keep the values of diagonal d + ORING
    double* ibz = A.IB + ((size_t)(d % ORING) * n + i) * 16 * MS2;
    for (int e = tid; e < 16 * MS2; e += OT) ibz[e] = 0.0;
    for (int e = tid; e < MS2; e += OT) A.IBS[((size_t)(d % ORING) * n + i) * MS2 + e] = 0.0;
    return;
  }

  // ---- 2: Qb-bar(i,j) -------------------------------------------------------------------------------------------------------------------------
  // the ring slot of this cell holds what closing cells pushed: adjoints of DD / GI / D1 / D2T stored at (i-1, j+1)
  const bool dressed = MI >= 2 && i >= 1 && j <= n - 2;
  const int nLm = dressed ? t.loff[i] - t.loff[i - 1] : 0, nRn = dressed ? t.roff[j + 2] - t.roff[j + 1] : 0;
  const int RDS = ML * MR + MS2 + ML * MS + MR * MS;
  // scratch record of the cell (PART 0 -> PART 1): Qb-bar | DD-bar | G | H1 | H2 | sum I | SB-bar | flag
  const int SCRS = scr_size(MS, ML, MR, nps);
  double* scr = A.SC + ((size_t)(d % SRING) * n + i) * SCRS;
  double *scr_ab = scr, *scr_ddb = scr_ab + ML * MR, *scr_go = scr_ddb + ML * MR, *scr_h1 = scr_go + 16 * MS2, *scr_h2 = scr_h1 + 4 * MS2,
         *scr_ibsum = scr_h2 + 4 * MS2, *scr_sbb = scr_ibsum + MS2, *scr_flag = scr_sbb + nps * MS2;
  if constexpr (PART == 1) {
    for (int e = tid; e < ML * MR; e += OT) { ab[e] = scr_ab[e]; ddb[e] = scr_ddb[e]; }
    for (int e = tid; e < 16 * MS2; e += OT) go[e] = scr_go[e];
    for (int e = tid; e < 4 * MS2; e += OT) { h1[e] = scr_h1[e]; h2[e] = scr_h2[e]; }
    for (int e = tid; e < MS2; e += OT) ibsum[e] = scr_ibsum[e];
    for (int e = tid; e < nps * MS2; e += OT) sbb[e] = scr_sbb[e];
  }
  double* rd = A.RD + ((size_t)(d % ORING) * n + i) * RDS;
  if (PART == 0 && dressed) {
    const double *add = rd, *agi = rd + ML * MR, *ad1 = agi + MS2, *ad2 = ad1 + ML * MS;
    for (int e = tid; e < nLm * nRn; e += OT) {
      const int lst = e / nRn, rr = e % nRn;
      const int a = sLa[0][lst], c = sRc[2][rr];
      ddb[lst * MR + rr] = add[lst * MR + rr] + agi[a * MS + c] + ad1[lst * MS + c] + ad2[rr * MS + a];
    }
  }
  for (int e = tid; e < npair; e += OT) qbv[e] = b.QB[(size_t)(Li0 + e / nR) * RS + Rj0 + e % nR];
  __syncthreads();
  bool anyp = true;
  if constexpr (PART == 0) {
  if (dressed)
    for (int e = tid; e < RDS; e += OT) rd[e] = 0.0;  // consumed: the slot is clean for diagonal d - ORING
  {
    // stack / bulge terms: pulled from the I tables of the closing pairs (i0,j0) = (i-1-l1, j+1+l2), l1 = 0 or l2 = 0.
    // Bulges of size >= 2 do not see the inner nucleotides: one sum per BOND pair (s,t) over the slot-summed tables IBS,
    //   bb[s][t] = sum_l1 w_Bu(l1) sum_a' E(i0+1,i-1)[a',s] IBS(i0,j+1)[a',t] + sum_l2 w_Bu(l2) sum_c' IBS(i-1,j0)[s,c'] E(j+1,j0-1)[t,c']
    {
      const int eb = tid % nent, gb = tid / nent, ngb = OT / nent;
      const int s_ = eb / Sj1, t_ = eb % Sj1;
      double accb = 0.0;
      if (gb < ngb)
        for (int qq = gb; qq < 2 * (MI - 1); qq += ngb) {
          const int left = qq < MI - 1, len = 2 + (left ? qq : qq - (MI - 1));
          const int i0 = left ? i - 1 - len : i - 1, j0 = left ? j + 1 : j + 1 + len;
          if (i0 < 0 || j0 > n - 1) continue;
          const double* ibsr = A.IBS + ((size_t)((j0 - i0) % ORING) * n + i0) * MS2;
          double v = 0.0;
          if (left) {
            const int Sa_ = sigA(i0 + 1);
            for (int a = 0; a < Sa_; ++a) v += EA(i0 + 1, i - 1, a, s_) * ibsr[a * MS + t_];
          } else {
            const int Sc_ = sigB(j0);
            for (int c = 0; c < Sc_; ++c) v += ibsr[s_ * MS + c] * EB(j + 1, j0 - 1, t_, c);
          }
          accb += m.wbu[len] * v;
        }
      const double tot = group_total(part, accb, nent);
      if (tid < nent) am[tid] = tot;  // (Qm-bar is no longer needed)
      __syncthreads();
    }
    // stacks and size-1 bulges keep the identity of the inner pair (weights by slot): one thread per state pair
    const int e2 = tid % npair;
    const int ll = e2 / nR, rr = e2 % nR;
    const int s = sLa[1][ll], xp = sLx[1][ll];
    const int yp = sRy[1][rr], tt_ = sRc[1][rr];
    const bool pairable = m.pslot[xp * 4 + yp] >= 0;
    double acc = 0.0;
    if (tid < npair && pairable) {
      const int Pin_st = m.ptype[xp * 4 + yp];  // inner pair as (phi_k, phi_l)
      for (int qq = 0; qq < 3; ++qq) {
        const int l1 = qq == 1, l2 = qq == 2;
        if (l1 + l2 > MI) continue;
        const int i0 = i - 1 - l1, j0 = j + 1 + l2;
        if (i0 < 0 || j0 > n - 1) continue;
        const double* ib = A.IB + ((size_t)((j0 - i0) % ORING) * n + i0) * 16 * MS2;
        const int Sa_ = sigA(i0 + 1), Sc_ = sigB(j0);
        for (int sl = 0; sl < nps; ++sl) {
          const double w = m.wst[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][Pin_st];
          double v = 0.0;
          if (qq == 0) v = ib[sl * MS2 + s * MS + tt_];
          else if (qq == 1) {  // left bulge of size 1: sum_a' Tbar_{i-1}[a',s] I[x,y;a',t]
            for (int a = 0; a < Sa_; ++a) v += EA(i0 + 1, i - 1, a, s) * ib[sl * MS2 + a * MS + tt_];
            v *= m.wbu[1];
          } else {  // right bulge of size 1
            for (int c = 0; c < Sc_; ++c) v += ib[sl * MS2 + s * MS + c] * EB(j + 1, j0 - 1, tt_, c);
            v *= m.wbu[1];
          }
          acc += w * v;
        }
      }
      acc += am[s * Sj1 + tt_];
    }
    const double v = acc;
    anyp = __syncthreads_or(tid < npair && pairable) != 0;  // can any nucleotide of i pair with any of j?
    if (tid < npair) {
      double w = 0.0;
      if (pairable) {
        w = v + abs_[s * Sj1 + tt_];
        if (dressed) {
          // interior loops: Qb(i,j) enters through its dressed extension DD(i-1,j+1)[lst][rr] = sum T_{i-1}[lst][s] T_{j+1}[t][rr]
          // e^{-beta tmm[p(y',x')][y(rr)][x(lst)]} Qb[(s,x')][(y',t)]
          const int Pil = m.ptype[yp * 4 + xp];
          double u = 0.0;
          for (int lst = 0; lst < nLm; ++lst) {
            const double tl = TLm[lst * MS + s];
            if (tl == 0.0) continue;
            const int up = sLx[0][lst];
            double r2 = 0.0;
            for (int r = 0; r < nRn; ++r)
              r2 += TRn[tt_ * MR + r] * m.wtm[Pil][sRy[2][r]][up] * ddb[lst * MR + r];
            u += tl * r2;
          }
          w += u;
        }
      }
      ab[tid] = w;
      A.AB[(size_t)(Li0 + ll) * RS + Rj0 + rr] = w;
      part[tid] = w * qbv[tid];
    }
    __syncthreads();
    if (tid == 0 && bpp && d > 0) {
      double pr = 0.0;
      for (int e = 0; e < npair; ++e) pr += part[e];
      bpp[(size_t)i * n + j] = pr;
    }
    __syncthreads();
  }
  }
  OTICK(1);
  if constexpr (PART == 1) {
    anyp = scr_flag[0] != 0.0;
    __syncthreads();  // the scratch record is in shared memory
  }
  // usages of the inner-mismatch operators z2 at i-1 (role IL) and z1' at j+1 (role IR)
  if (PART == 1 && want_usage && dressed && anyp) {
    const int z2b = t.opstart[i - 1], nz2 = t.opstart[i] - z2b, z1b = t.opstart[j + 1], nz1 = t.opstart[j + 2] - z1b;
    for (int e = tid; e < nz2 + nz1; e += OT) {
      double u = 0.0;
      if (e < nz2) {
        const int z = z2b + e, lst = t.op_l[z], s = t.op_c[z], up = t.op_b[z];
        for (int ll = 0; ll < nL; ++ll) {
          if (sLa[1][ll] != s) continue;
          const int xp = sLx[1][ll];
          for (int rr = 0; rr < nR; ++rr) {
            const int yp = sRy[1][rr], tt_ = sRc[1][rr];
            if (m.pslot[xp * 4 + yp] < 0) continue;
            const int Pil = m.ptype[yp * 4 + xp];
            double r2 = 0.0;
            for (int r = 0; r < nRn; ++r)
              r2 += TRn[tt_ * MR + r] * m.wtm[Pil][sRy[2][r]][up] * ddb[lst * MR + r];
            u += r2 * qbv[ll * nR + rr];
          }
        }
        A.U[(size_t)ROLE_IL * A.nops + z] += t.op_x[z] * u;
      } else {
        const int z = z1b + (e - nz2), r = t.op_r[z], tt_ = t.op_a[z], vp = t.op_b[z];
        for (int rr = 0; rr < nR; ++rr) {
          if (sRc[1][rr] != tt_) continue;
          const int yp = sRy[1][rr];
          for (int ll = 0; ll < nL; ++ll) {
            const int xp = sLx[1][ll], s = sLa[1][ll];
            if (m.pslot[xp * 4 + yp] < 0) continue;
            const int Pil = m.ptype[yp * 4 + xp];
            double r2 = 0.0;
            for (int lst = 0; lst < nLm; ++lst)
              r2 += TLm[lst * MS + s] * m.wtm[Pil][vp][sLx[0][lst]] * ddb[lst * MR + r];
            u += r2 * qbv[ll * nR + rr];
          }
        }
        A.U[(size_t)ROLE_IR * A.nops + z] += t.op_x[z] * u;
      }
    }
  }

  const int Sa = t.sig[p], Sc = t.sig[j];  // a' in Sigma_{i+1}, c' in Sigma_j
  const bool has_loop = q > p;            // positions i+1 and j-1 are distinct unpaired positions (always true for min_hairpin >= 3)
  if constexpr (PART == 0) {
  OTICK(2);
  // ---- 3: I(i,j)[slot][a'][c'], G[u,v][a'][c'], H, H1, H2 ----------------------------------------------------------------------------------
  double* ibo = A.IB + ((size_t)(d % ORING) * n + i) * 16 * MS2;
  // I[slot][a'][c'] = sum_{z at i: b = x, c = a'} sum_{z' at j: b = y, a = c'} x_z x_z' Qb-bar[l(z)][r(z')], in two steps through the dense
  // cores: T1[x][a'][r] = sum_{l: x(l) = x} T_i[l][a'] Qb-bar[l][r], then I = sum_{r: y(r) = y} T_j[c'][r] T1[x][a'][r]
  double* t1 = y;  // (Y and Z1 are not in use yet; T1 needs 4 MS MR <= ML MR + ML MS doubles, see oplan)
  for (int e = tid; e < 4 * MS * nR; e += OT) {
    const int x = e / (MS * nR), ap = (e / nR) % MS, r = e % nR;
    double v = 0.0;
    if (ap < Sa)
      for (int l = 0; l < nL; ++l)
        if (sLx[1][l] == x) v += TLi[l * MS + ap] * ab[l * nR + r];
    t1[e] = v;
  }
  __syncthreads();
  for (int e = tid; e < 16 * MS2; e += OT) {
    const int sl = e / MS2, ap = (e % MS2) / MS, cp = e % MS;
    double v = 0.0;
    if (sl < nps && ap < Sa && cp < Sc) {
      const int x = m.slot_x[sl], yy = m.slot_y[sl];
      const double* tp = t1 + (x * MS + ap) * nR;
      for (int r = 0; r < nR; ++r)
        if (sRy[1][r] == yy) v += TRj[cp * MR + r] * tp[r];
    }
    if (sl < nps) ibs[e] = v;
    ibo[e] = v;
  }
  __syncthreads();
  for (int e = tid; e < 16 * MS2; e += OT) {
    const int uv = e / MS2, r = e % MS2;
    double v = 0.0;
    for (int sl = 0; sl < nps; ++sl) v += ibs[sl * MS2 + r] * m.wtm[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][uv >> 2][uv & 3];
    go[e] = v;
  }
  for (int e = tid; e < MS2; e += OT) {
    double v = 0.0;
    for (int sl = 0; sl < nps; ++sl) v += ibs[sl * MS2 + e];
    ibsum[e] = v;  // adjoint of Bl / Br / the multiloop closure: they enter `inner` of every pairable slot
    A.IBS[((size_t)(d % ORING) * n + i) * MS2 + e] = v;
  }
  for (int e = tid; e < nps * MS2; e += OT) {
    // adjoint of SB[a'][slot'][c'] (stored [slot'][a'][c']):  sum_slot wst[P][P'] I[slot]
    const int sl2 = e / MS2, r = e % MS2;
    const int P2 = m.ptype[m.slot_x[sl2] * 4 + m.slot_y[sl2]];
    double v = 0.0;
    for (int sl = 0; sl < nps; ++sl) v += m.wst[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][P2] * ibs[sl * MS2 + r];
    sbb[e] = v;
  }
  __syncthreads();
  // Loop-side operators contracted with G through the dense cores T_p[lst][c], T_q[a][r] (shared memory only):
  //   H1[u][a][a2'] = sum_{z2' at q: a = a2'} x' G[u,b(z2')][a][c(z2')] = sum_r T_q[a2'][r] G[u,y(r)][a][c(r)]        (adjoint of Z1)
  //   H2[v][c1][c'] = sum_{z1 at p: c = c1} x G[b(z1),v][a(z1)][c']     = sum_lst T_p[lst][c1] G[x(lst),v][a(lst)][c']  (adjoint of Z2)
  //   H[c1][a2']    = sum_lst T_p[lst][c1] H1[x(lst)][a(lst)][a2']                                                    (adjoint of XE)
  {
    const int nLp_ = t.loff[p + 1] - t.loff[p], nRq_ = t.roff[q + 1] - t.roff[q];
    for (int e = tid; e < 8 * MS2; e += OT) {
      const int which = e / (4 * MS2), r = e % (4 * MS2);
      const int uv = r / MS2, x1 = (r % MS2) / MS, x2 = r % MS;
      double v = 0.0;
      if (has_loop) {
        if (which == 0) {
          for (int rr = 0; rr < nRq_; ++rr) v += TRq[x2 * MR + rr] * go[(uv * 4 + sRy[0][rr]) * MS2 + x1 * MS + sRc[0][rr]];
        } else {
          for (int lst = 0; lst < nLp_; ++lst) v += TLp[lst * MS + x1] * go[(sLx[2][lst] * 4 + uv) * MS2 + sLa[2][lst] * MS + x2];
        }
      }
      (which == 0 ? h1 : h2)[r] = v;
    }
    __syncthreads();
    for (int e = tid; e < MS2; e += OT) {
      const int c1 = e / MS, a2p = e % MS;
      double v = 0.0;
      if (has_loop)
        for (int lst = 0; lst < nLp_; ++lst) v += TLp[lst * MS + c1] * h1[(sLx[2][lst] * MS + sLa[2][lst]) * MS + a2p];
      h[e] = v;
    }
  }
  __syncthreads();

    // hand the cell over to PART 1
    for (int e = tid; e < ML * MR; e += OT) { scr_ab[e] = e < npair ? ab[(e / nR) * nR + e % nR] : 0.0; scr_ddb[e] = ddb[e]; }
    for (int e = tid; e < 16 * MS2; e += OT) scr_go[e] = go[e];
    for (int e = tid; e < 4 * MS2; e += OT) { scr_h1[e] = h1[e]; scr_h2[e] = h2[e]; }
    for (int e = tid; e < MS2; e += OT) scr_ibsum[e] = ibsum[e];
    for (int e = tid; e < nps * MS2; e += OT) scr_sbb[e] = sbb[e];
    if (tid == 0) scr_flag[0] = anyp ? 1.0 : 0.0;
  }
  OTICK(3);
  // ---- 4: this cell as closing pair ---------------------------------------------------------------------------------------------------------
  const int Sp1 = t.sig[p + 1], Sq = t.sig[q];  // bonds after i+1 / before j-1: XE, H are Sp1 x Sq
  const int nLp = t.loff[p + 1] - t.loff[p], nRq = t.roff[q + 1] - t.roff[q];
  const int Lp0 = t.loff[p], Rq0 = t.roff[q];
  double* xa = A.XA + ((size_t)(d % XRING) * n + i) * XU * MS2;
  double* xb = A.XB + ((size_t)(d % XRING) * n + i) * XU * MS2;
  if constexpr (PART == 0) {
  // 4a hairpin interior E(p+1,q-1): its adjoint is w_H(d-1) H (single writer: plain store into the transposed table)
  {
    const double wh = t.wh[d - 1];
    for (int e = tid; e < Sp1 * Sq; e += OT) {
      const int cz = e / Sq, aw = e % Sq;
      A.AET[(size_t)(t.off[q] + aw) * S + t.off[p + 1] + cz] = wh * h[cz * MS + aw];
    }
  }
  // 4b adjoint row / column recursions of the interior-loop bodies (u = 4..30):
  //      XA_u(i,j) = w_In(u) H + Tbar_{i+1}^T XA_{u+1}(i-1,j)          XB_u(i,j) = w_In(u) H + XB_{u+1}(i,j+1) Tbar_{j-1}^T
  {
    const double* xa1 = i >= 1 ? A.XA + ((size_t)((d + 1) % XRING) * n + (i - 1)) * XU * MS2 : nullptr;
    const double* xb1 = j + 1 <= n - 1 ? A.XB + ((size_t)((d + 1) % XRING) * n + i) * XU * MS2 : nullptr;
    for (int e = tid; e < XU * MS2; e += OT) {
      const int u4 = e / MS2, cz = (e % MS2) / MS, aw = e % MS, u = u4 + 4;
      double va = 0.0, vb = 0.0;
      if (cz < Sp1 && aw < Sq) {
        const double w = u <= MI ? m.win[u] * h[cz * MS + aw] : 0.0;
        va = vb = w;
        if (u4 + 1 < XU) {
          if (xa1) {
            const double* src = xa1 + (u4 + 1) * MS2 + aw;
            for (int a = 0; a < t.sig[p]; ++a) va += t.Tbar[((size_t)p * MS + a) * MS + cz] * src[a * MS];
          }
          if (xb1) {
            const double* src = xb1 + (u4 + 1) * MS2 + cz * MS;
            for (int c = 0; c < t.sig[j]; ++c) vb += src[c] * t.Tbar[((size_t)q * MS + aw) * MS + c];
          }
        }
      }
      xa[e] = va;
      xb[e] = vb;
    }
  }
  __syncthreads();
    OTICK(4);
    return;
  }
  OTICK(4);
  // 4c pushes of the generic interior loops (l1, l2 >= 2).  All terms of X_u(i,j) have the inner span d-2-u.
  if (MI >= 4) {
    // row recursion, new term GI(i+3, l) E(l+2,j-2), l = j+1-u:  adjoint of GI into the ring slot of cell (i+3,l); E-bar of the right stretch
    for (int e = tid; e < XU * MS2; e += OT) {
      const int u4 = e / MS2, x1 = (e % MS2) / MS, x2 = e % MS, u = u4 + 4;
      if (d - 2 - u < mh1) continue;
      const int l = j + 1 - u, k = i + 3;  // inner pair (k,l): l1 = 2, l2 = u-2
      const int Sk1 = Sp1 /* Sigma_{k-1} = Sigma_{i+2} */, Sl2 = sigB(l + 2);
      const double* xau = xa + u4 * MS2;
      // AGI(k,l)[s2 = x1][t2 = x2] += sum_aw XA_u[s2][aw] E(l+2,j-2)[t2][aw]
      if (x1 < Sk1 && x2 < Sl2) {
        double v = 0.0;
        for (int aw = 0; aw < Sq; ++aw) v += xau[x1 * MS + aw] * EB(l + 2, j - 2, x2, aw);
        double* rdk = A.RD + ((size_t)((l - k) % ORING) * n + k) * RDS + ML * MR;
        rdk[x1 * MS + x2] += v;
      }
      // E-bar(l+2, j-2)[t2 = x1][aw = x2] += sum_s2 GI(k,l)[s2][t2] XA_u[s2][aw]       (length u-4 >= 1)
      if (want_usage && u > 4 && x1 < Sl2 && x2 < Sq) {
        const double* gi = b.GI + (size_t)offA(k - 1) * S + offB(l + 2) + x1;
        double v = 0.0;
        for (int s2 = 0; s2 < Sk1; ++s2) v += gi[(size_t)s2 * S] * xau[s2 * MS + x2];
        A.AES[(((size_t)AES_XR * n + (l + 2)) * SLEN + (u - 4)) * MS2 + x1 * MS + x2] += v;
      }
    }
    // column recursion, new term E(i+2,k-2) GI(k, j-3), k = i+u-1:  E-bar of the left stretch (length u-4 >= 1)
    if (want_usage)
      for (int e = tid; e < XU * MS2; e += OT) {
        const int u4 = e / MS2, cz = (e % MS2) / MS, s2 = e % MS, u = u4 + 4;
        if (u == 4 || d - 2 - u < mh1) continue;
        const int k = i + u - 1, l = j - 3;
        if (cz >= Sp1 || s2 >= sigA(k - 1)) continue;
        const double* gi = b.GI + (size_t)(offA(k - 1) + s2) * S + offB(l + 2);  // columns: bonds of position l+2 = j-1
        const double* xbu = xb + u4 * MS2 + cz * MS;
        double v = 0.0;
        for (int aw = 0; aw < Sq; ++aw) v += xbu[aw] * gi[aw];
        A.AES[(((size_t)AES_XL * n + (i + 2)) * SLEN + (u - 4)) * MS2 + cz * MS + s2] += v;
      }
  }
  OTICK(5);
  if (!anyp) return;  // no nucleotide of i pairs with one of j: G = H = 0, only the chains above pass through this cell
  // 4d pushes of the l1 = 1 / l2 = 1 / 1x1 interior loops
  if (MI >= 2) {
    // 1 x 1: inner pair (i+2, j-2), DD(p,q) enters Y with w_In(2)
    if (d - 4 >= mh1) {
      double* rdk = A.RD + ((size_t)((d - 4) % ORING) * n + (i + 2)) * RDS;
      for (int e = tid; e < nLp * nRq; e += OT) {
        const int lst = e / nRq, r = e % nRq;
        rdk[lst * MR + r] += m.win[2] * go[(sLx[2][lst] * 4 + sRy[0][r]) * MS2 + sLa[2][lst] * MS + sRc[0][r]];
      }
    }
    // l1 = 1, l2 = 2..lmax1: Z1[lst][c2] = sum_l2 w_In(1+l2) sum_u D1(p; l+2)[lst][u] E(l+2,q-1)[u][c2],  l = q - l2; inner pair (i+2, l)
    // l2 = 1, l1 = 2..lmax2: Z2[a2][r] = sum_l1 w_In(l1+1) sum_s E(p+1,k-2)[a2][s] D2(k-1; q)[s][r],  k = p + l1; inner pair (k, j-2)
    // (all (l, entry) items of the four pushes are independent: one flat loop over the threads)
    const int lmax1 = min(MI - 1, q - mh1 - (p + 1)), lmax2 = min(MI - 1, (q - 1) - mh1 - p);
    const int n1 = max(lmax1 - 1, 0), n2 = max(lmax2 - 1, 0);
    const int e1 = n1 * nLp * MS, e2 = e1 + n2 * nRq * MS, e3 = e2 + (want_usage ? n1 * MS2 : 0), e4 = e3 + (want_usage ? n2 * MS2 : 0);
    for (int e = tid; e < e4; e += OT) {
      if (e < e1) {
        const int l2 = 2 + e / (nLp * MS), lst = (e / MS) % nLp, u = e % MS, l = q - l2;
        if (u >= sigB(l + 2)) continue;
        const double* hz = h1 + (sLx[2][lst] * MS + sLa[2][lst]) * MS;  // Z1-bar[lst][c2] = H1[x(lst)][a(lst)][c2]
        double v = 0.0;
        for (int c2 = 0; c2 < Sq; ++c2) v += hz[c2] * EB(l + 2, q - 1, u, c2);
        double* rdk = A.RD + ((size_t)((l - (i + 2)) % ORING) * n + (i + 2)) * RDS + ML * MR + MS2;  // AD1[lst][u] of cell (i+2, l)
        rdk[lst * MS + u] += m.win[1 + l2] * v;
      } else if (e < e2) {
        const int f = e - e1, l1 = 2 + f / (nRq * MS), r = (f / MS) % nRq, s_ = f % MS, k = p + l1;
        if (s_ >= sigA(k - 1)) continue;
        const double* hz = h2 + (sRy[0][r] * MS) * MS + sRc[0][r];  // Z2-bar[a2][r] = H2[y(r)][a2][c(r)]
        double v = 0.0;
        for (int a2 = 0; a2 < Sp1; ++a2) v += EA(p + 1, k - 2, a2, s_) * hz[a2 * MS];
        double* rdk = A.RD + ((size_t)(((j - 2) - k) % ORING) * n + k) * RDS + ML * MR + MS2 + ML * MS;  // AD2[r][s] of cell (k, j-2)
        rdk[r * MS + s_] += m.win[l1 + 1] * v;
      } else if (e < e3) {
        // E-bar(l+2, q-1)[u][c2] += w sum_lst D1[lst][u] Z1-bar[lst][c2]        (length l2 - 2 >= 1)
        const int f = e - e2, l2 = 2 + f / MS2, u = (f % MS2) / MS, c2 = f % MS, l = q - l2;
        if (l2 == 2 || u >= sigB(l + 2) || c2 >= Sq) continue;
        double v = 0.0;
        for (int lst = 0; lst < nLp; ++lst)
          v += b.D1[(size_t)(Lp0 + lst) * S + offB(l + 2) + u] * h1[(sLx[2][lst] * MS + sLa[2][lst]) * MS + c2];
        A.AES[(((size_t)AES_Z1R * n + (l + 2)) * SLEN + (l2 - 2)) * MS2 + u * MS + c2] += m.win[1 + l2] * v;
      } else {
        // E-bar(p+1, k-2)[a2][s] += w sum_r Z2-bar[a2][r] D2(k-1; q)[s][r]      (length l1 - 2 >= 1)
        const int f = e - e3, l1 = 2 + f / MS2, a2 = (f % MS2) / MS, s_ = f % MS, k = p + l1;
        if (l1 == 2 || a2 >= Sp1 || s_ >= sigA(k - 1)) continue;
        double v = 0.0;
        for (int r = 0; r < nRq; ++r)
          v += h2[(sRy[0][r] * MS + a2) * MS + sRc[0][r]] * b.D2T[(size_t)(Rq0 + r) * S + offA(k - 1) + s_];
        A.AES[(((size_t)AES_Z2L * n + (p + 1)) * SLEN + (l1 - 2)) * MS2 + a2 * MS + s_] += m.win[l1 + 1] * v;
      }
    }
  }
  OTICK(6);
  if (!want_usage) return;
  const int offp_ = offA(p), offj_ = offB(j), offp1_ = offA(p + 1), offq_ = offB(q);
  // 4e stretch adjoints of the bulges of size >= 2:  Bl = .. + sum_l1 w_Bu(l1) E(p,k-1) Qbs(k,q),  Br = sum_l2 w_Bu(l2) Qbs(p,l) E(l+1,q)
  {
    const int lmax = min(MI, q - mh1 - p);
    for (int e = tid; e < (lmax >= 2 ? (lmax - 1) * 2 * MS2 : 0); e += OT) {
      const int side = e / ((lmax - 1) * MS2), r = e % ((lmax - 1) * MS2);
      const int len = 2 + r / MS2, x1 = (r % MS2) / MS, x2 = r % MS;
      if (side == 0) {
        const int k = p + len;  // E(p,k-1)[a1 = x1][s = x2]
        if (x1 >= Sa || x2 >= sigA(k)) continue;
        const double* qs = b.QBS + (size_t)(offA(k) + x2) * S + offj_;
        double v = 0.0;
        for (int c1 = 0; c1 < Sc; ++c1) v += ibsum[x1 * MS + c1] * qs[c1];
        A.AES[(((size_t)AES_BL * n + p) * SLEN + len) * MS2 + x1 * MS + x2] += m.wbu[len] * v;
      } else {
        const int l = q - len;  // E(l+1,q)[u = x1][c1 = x2]
        if (x1 >= sigB(l + 1) || x2 >= Sc) continue;
        double v = 0.0;
        for (int a1 = 0; a1 < Sa; ++a1) v += b.QBS[(size_t)(offp_ + a1) * S + offB(l + 1) + x1] * ibsum[a1 * MS + x2];
        A.AES[(((size_t)AES_BR * n + (l + 1)) * SLEN + len) * MS2 + x1 * MS + x2] += m.wbu[len] * v;
      }
    }
  }
  OTICK(7);
  // 4f forward quantities of this cell, recomputed from the stored tables exactly as the inside pass builds them
  {
    const int lmaxB = min(MI, q - mh1 - p);
    const int lmaxZ1 = min(MI - 1, q - mh1 - (p + 1)), lmaxZ2 = min(MI - 1, (q - 1) - mh1 - p);
    for (int e = tid; e < Sp1 * Sq; e += OT) xe[(e / Sq) * MS + e % Sq] = b.XE[(size_t)(offp1_ + e / Sq) * S + offq_ + e % Sq];
    // Bl, Br [a1 < Sa][c1 < Sc], Z1[lst][c2 < Sq], Z2[a2 < Sp1][r]: one thread per entry, weighted dot products over the bonds of
    // the <= 29 band positions (offsets from the shared windows, so the loads of different positions are independent)
    const int nb = Sa * Sc, nz1 = nLp * Sq, nz2 = Sp1 * nRq;
    for (int e = tid; e < 2 * nb + nz1 + nz2; e += OT) {
      const double *A_, *B_, *wt;
      int lo, hi, near_i, base_pos, sgn;  // positions lo..hi, weight wt[sgn * (pos - base_pos)]
      double v = 0.0;
      double* out;
      if (e < nb) {
        const int a1 = e / Sc, c1 = e % Sc;
        v = m.wac * b.M2[(size_t)(offp_ + a1) * S + offj_ + c1];
        A_ = b.EM + (size_t)(offp_ + a1) * S; B_ = b.QBST + (size_t)(offj_ + c1) * S;
        lo = p + 2; hi = p + lmaxB; near_i = 1; wt = m.wbu; base_pos = p; sgn = 1;  // k = p + l1
        out = bl + a1 * MS + c1;
      } else if (e < 2 * nb) {
        const int a1 = (e - nb) / Sc, c1 = (e - nb) % Sc;
        A_ = b.QBS + (size_t)(offp_ + a1) * S; B_ = b.EMT + (size_t)(offj_ + c1) * S;
        lo = q - lmaxB + 1; hi = q - 1; near_i = 0; wt = m.wbu; base_pos = j; sgn = -1;  // pos = l + 1, l2 = j - pos
        out = br + a1 * MS + c1;
      } else if (e < 2 * nb + nz1) {
        const int f = e - 2 * nb, lst = f / Sq, c2 = f % Sq;
        A_ = b.D1 + (size_t)(Lp0 + lst) * S; B_ = b.EMT + (size_t)(offq_ + c2) * S;
        lo = q - lmaxZ1 + 2; hi = q; near_i = 0; wt = m.win; base_pos = j + 2; sgn = -1;  // pos = l + 2, weight w_In(1 + l2) = win[j + 2 - pos]
        out = z1 + lst * MS + c2;
      } else {
        const int f = e - 2 * nb - nz1, a2 = f / nRq, r = f % nRq;
        A_ = b.EM + (size_t)(offp1_ + a2) * S; B_ = b.D2T + (size_t)(Rq0 + r) * S;
        lo = p + 1; hi = p + lmaxZ2 - 1; near_i = 1; wt = m.win; base_pos = p - 2; sgn = 1;  // pos = k - 1, weight w_In(l1 + 1) = win[pos + 2 - p]
        out = z2 + a2 * MR + r;
      }
#pragma unroll 4
      for (int pos = lo; pos <= hi; ++pos) {
        const int o = near_i ? offA(pos) : offB(pos), sg = near_i ? sigA(pos) : sigB(pos);
        double s = 0.0;
        for (int kb = o; kb < o + sg; ++kb) s += A_[kb] * B_[kb];
        v += wt[sgn * (pos - base_pos)] * s;
      }
      *out = v;
    }
    // SB[slot'][a1][c1]: stack + size-1 bulges (the inner pair keeps its identity)
    for (int e = tid; e < nps * Sa * Sc; e += OT) {
      const int sl = e / (Sa * Sc), a1 = (e % (Sa * Sc)) / Sc, c1 = e % Sc;
      const int xp = m.slot_x[sl], yp = m.slot_y[sl];
      const int lst = t.lsidx[((size_t)p * MS + a1) * 4 + xp], r = t.rsidx[((size_t)q * 4 + yp) * MS + c1];
      double v = 0.0;
      if (q - p >= mh1 && lst >= 0 && r >= 0) v = b.QB[(size_t)(Lp0 + lst) * RS + Rq0 + r];
      if (MI >= 1 && q - (p + 1) >= mh1) {
        double s1 = 0.0, s2 = 0.0;
        if (r >= 0)
          for (int l2 = t.loff[p + 1]; l2 < t.loff[p + 2]; ++l2)
            if (t.ls_x[l2] == xp) s1 += t.Tbar[((size_t)p * MS + a1) * MS + t.ls_a[l2]] * b.QB[(size_t)l2 * RS + Rq0 + r];
        if (lst >= 0)
          for (int r2 = t.roff[q - 1]; r2 < t.roff[q]; ++r2)
            if (t.rs_y[r2] == yp) s2 += b.QB[(size_t)(Lp0 + lst) * RS + r2] * t.Tbar[((size_t)q * MS + t.rs_c[r2]) * MS + c1];
        v += m.wbu[1] * (s1 + s2);
      }
      sb[sl * MS2 + a1 * MS + c1] = v;
    }
  }
  __syncthreads();
  {
    // Y[lst][r] = w_In(2) DD(p,q) + sum_cz T_p[lst][cz] (Z2[cz][r] + sum_aw XE[cz][aw] T_q[aw][r]) + sum_aw Z1[lst][aw] T_q[aw][r]
    const bool v11 = MI >= 2 && d - 4 >= mh1;
    for (int e = tid; e < nLp * nRq; e += OT) {
      const int lst = e / nRq, r = e % nRq;
      double v = v11 ? m.win[2] * b.DD[(size_t)(Lp0 + lst) * RS + Rq0 + r] : 0.0;
      for (int cz = 0; cz < Sp1; ++cz) {
        const double tl = TLp[lst * MS + cz];
        if (tl == 0.0) continue;
        double s = z2[cz * MR + r];
        for (int aw = 0; aw < Sq; ++aw) s += xe[cz * MS + aw] * TRq[aw * MR + r];
        v += tl * s;
      }
      for (int aw = 0; aw < Sq; ++aw) v += z1[lst * MS + aw] * TRq[aw * MR + r];
      y[lst * MR + r] = v;
    }
  }
  __syncthreads();
  // inner[slot][a1][c1] = Bl + Br + sum_slot' wst[P][P'] SB[slot'] + sum_{(a1,u),(v,c1)} wtm[P][u][v] Y
  for (int e = tid; e < nps * Sa * Sc; e += OT) {
    const int sl = e / (Sa * Sc), a1 = (e % (Sa * Sc)) / Sc, c1 = e % Sc;
    const int P = m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]];
    double v = bl[a1 * MS + c1] + br[a1 * MS + c1];
    for (int s2 = 0; s2 < nps; ++s2) v += m.wst[P][m.ptype[m.slot_x[s2] * 4 + m.slot_y[s2]]] * sb[s2 * MS2 + a1 * MS + c1];
    for (int lst = 0; lst < nLp; ++lst) {
      if (sLa[2][lst] != a1) continue;
      const int u = sLx[2][lst];
      for (int r = 0; r < nRq; ++r)
        if (sRc[0][r] == c1) v += m.wtm[P][u][sRy[0][r]] * y[lst * MR + r];
    }
    inn[sl * MS2 + a1 * MS + c1] = v;
  }
  __syncthreads();
  OTICK(8);
  // ---- usages ----------------------------------------------------------------------------------------------------------------------------------
  {
    const int zi0 = t.opstart[i], ni = t.opstart[i + 1] - zi0, zj0 = t.opstart[j], nj = t.opstart[j + 1] - zj0;
    const int zp0 = t.opstart[p], np_ = t.opstart[p + 1] - zp0, zq0 = t.opstart[q], nq = t.opstart[q + 1] - zq0;
    const size_t no = A.nops;
    for (int e = tid; e < ni + nj + 2 * np_ + 2 * nq; e += OT) {
      if (e < ni) {
        // pair end i:  x_z sum_{z' at j} x_z' Qb-bar[l(z)][r(z')] inner[slot(x,y)][c(z)][a(z')]
        const int z = zi0 + e, x = t.op_b[z];
        double u = 0.0;
        for (int zz = zj0; zz < zj0 + nj; ++zz) {
          const int sl = m.pslot[x * 4 + t.op_b[zz]];
          if (sl >= 0) u += t.op_x[zz] * ab[t.op_l[z] * nR + t.op_r[zz]] * inn[sl * MS2 + t.op_c[z] * MS + t.op_a[zz]];
        }
        A.U[(size_t)ROLE_PL * no + z] += t.op_x[z] * u;
      } else if (e < ni + nj) {
        const int zz = zj0 + (e - ni), yy = t.op_b[zz];
        double u = 0.0;
        for (int z = zi0; z < zi0 + ni; ++z) {
          const int sl = m.pslot[t.op_b[z] * 4 + yy];
          if (sl >= 0) u += t.op_x[z] * ab[t.op_l[z] * nR + t.op_r[zz]] * inn[sl * MS2 + t.op_c[z] * MS + t.op_a[zz]];
        }
        A.U[(size_t)ROLE_PR * no + zz] += t.op_x[zz] * u;
      } else if (e < ni + nj + np_) {
        // closing mismatch at p = i+1 (hairpins and interior loops with l1 >= 2):
        //   x_z1 ( sum_r G[u, y(r)][a1][c(r)] Z2[cz][r] + sum_aw XE[cz][aw] H1[u][a1][aw] )
        const int z1_ = zp0 + (e - ni - nj), a1 = t.op_a[z1_], u_ = t.op_b[z1_], cz = t.op_c[z1_];
        double u = 0.0;
        if (has_loop) {
          for (int r = 0; r < nRq; ++r)
            u += go[(u_ * 4 + sRy[0][r]) * MS2 + a1 * MS + sRc[0][r]] * z2[cz * MR + r];
          for (int aw = 0; aw < Sq; ++aw) u += xe[cz * MS + aw] * h1[(u_ * MS + a1) * MS + aw];
        }
        A.U[(size_t)ROLE_CL * no + z1_] += t.op_x[z1_] * u;
      } else if (e < ni + nj + np_ + nq) {
        // closing mismatch at q = j-1:  x_z2' ( sum_cz XE[cz][aw] H2[v][cz][c1] + sum_lst G[x(lst), v][a(lst)][c1] Z1[lst][aw] )
        const int z2_ = zq0 + (e - ni - nj - np_), aw = t.op_a[z2_], v_ = t.op_b[z2_], c1 = t.op_c[z2_];
        double u = 0.0;
        if (has_loop) {
          for (int cz = 0; cz < Sp1; ++cz) u += xe[cz * MS + aw] * h2[(v_ * MS + cz) * MS + c1];
          for (int lst = 0; lst < nLp; ++lst)
            u += go[(sLx[2][lst] * 4 + v_) * MS2 + sLa[2][lst] * MS + c1] * z1[lst * MS + aw];
        }
        A.U[(size_t)ROLE_CR * no + z2_] += t.op_x[z2_] * u;
      } else if (e < ni + nj + 2 * np_ + nq) {
        // size-1 left bulge at p (unpaired, no mismatch): x_z w_Bu(1) sum_{slot',c1} SB-bar[slot'][a1][c1] Qb(p+1,q)[(s,x')][(y',c1)]
        const int z = zp0 + (e - ni - nj - np_ - nq), a1 = t.op_a[z], s = t.op_c[z];
        double u = 0.0;
        if (MI >= 1 && q - (p + 1) >= mh1)
          for (int sl = 0; sl < nps; ++sl) {
            const int lst = t.lsidx[((size_t)(p + 1) * MS + s) * 4 + m.slot_x[sl]];
            if (lst < 0) continue;
            for (int c1 = 0; c1 < Sc; ++c1) {
              const int r = t.rsidx[((size_t)q * 4 + m.slot_y[sl]) * MS + c1];
              if (r >= 0) u += sbb[sl * MS2 + a1 * MS + c1] * b.QB[(size_t)(t.loff[p + 1] + lst) * RS + Rq0 + r];
            }
          }
        A.U[(size_t)ROLE_B1L * no + z] += t.op_x[z] * m.wbu[1] * u;
      } else {
        // size-1 right bulge at q: x_z w_Bu(1) sum_{slot',a1} SB-bar[slot'][a1][c1] Qb(p,q-1)[(a1,x')][(y',t)]
        const int z = zq0 + (e - ni - nj - 2 * np_ - nq), tt_ = t.op_a[z], c1 = t.op_c[z];
        double u = 0.0;
        if (MI >= 1 && q - (p + 1) >= mh1)
          for (int sl = 0; sl < nps; ++sl) {
            const int r = t.rsidx[((size_t)(q - 1) * 4 + m.slot_y[sl]) * MS + tt_];
            if (r < 0) continue;
            for (int a1 = 0; a1 < Sa; ++a1) {
              const int lst = t.lsidx[((size_t)p * MS + a1) * 4 + m.slot_x[sl]];
              if (lst >= 0) u += sbb[sl * MS2 + a1 * MS + c1] * b.QB[(size_t)(Lp0 + lst) * RS + t.roff[q - 1] + r];
            }
          }
        A.U[(size_t)ROLE_B1R * no + z] += t.op_x[z] * m.wbu[1] * u;
      }
    }
  }
  OTICK(9);
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------------------------------------------
size_t cdz_outside_carve(const cdz_tt* tt, void* base, Adj* out) {
  const size_t n = tt->n, S = tt->S, LS = tt->LS, RS = tt->RS, MS = tt->MS, MS2 = MS * MS, nops = tt->ops.size();
  const size_t ML = tt->maxL, MR = tt->maxR;
  Adj A;
  memset(&A, 0, sizeof(A));
  size_t used = 0;
  auto take = [&](size_t count) {
    used = (used + 255) & ~size_t(255);
    double* p = base ? (double*)((char*)base + used) : nullptr;
    used += count * sizeof(double);
    return p;
  };
  A.ML = (int)ML; A.MR = (int)MR; A.nops = nops;
  A.AM2 = take(S * S); A.AM2T = take(S * S); A.AML = take(S * S); A.AM1T = take(S * S); A.AET = take(S * S);
  A.QM1 = take(S * S); A.QMT = take(S * S);
  A.AB = take(LS * RS);
  A.AX = take((n + 1) * MS); A.AXB = take(S);
  A.IB = take((size_t)ORING * n * 16 * MS2);
  A.IBS = take((size_t)ORING * n * MS2);
  A.RD = take((size_t)ORING * n * (ML * MR + MS2 + ML * MS + MR * MS));
  A.XA = take((size_t)XRING * n * XU * MS2); A.XB = take((size_t)XRING * n * XU * MS2);
  A.SC = take((size_t)SRING * n * scr_size((int)MS, (int)ML, (int)MR, 16));
  A.AES = take((size_t)AES_NROLE * n * SLEN * MS2);
  A.U = take((size_t)NROLE * nops);
  A.status = (int*)take(8);
  if (out) *out = A;
  return (used + 255) & ~size_t(255);
}

int cdz_launch_outside(cdz_tables* t, const Adj& A, size_t ws_bytes, double* bpp_dev, double* base_dev, double* codon_dev, cudaStream_t st) {
  const cdz_tt* tt = t->tt;
  const int n = tt->n, NB = tt->NB;
  const int want_usage = 1;  // the unpaired diagonal of bpp also comes from the usages (independent of the pair sums)
  CDZ_CUDA(cudaMemsetAsync(A.AM2, 0, ws_bytes, st));  // AM2 is the first array of the workspace
  if (bpp_dev) CDZ_CUDA(cudaMemsetAsync(bpp_dev, 0, (size_t)n * n * sizeof(double), st));
  transpose_kernel<<<dim3(NB, NB), 256, 0, st>>>(t->h.tab.QM1T, A.QM1, tt->S, 1);
  transpose_kernel<<<dim3(NB, NB), 256, 0, st>>>(t->h.tab.QM, A.QMT, tt->S, 0);
  oext_kernel<<<1, 1024, 0, st>>>(t->d_ctx, A);
  const OPlan pl = oplan(tt->MS, tt->maxL, tt->maxR, t->model->c.nps);
  const size_t smem = sizeof(double) * pl.total;
  const bool small = tt->MS <= 4;  // compile-time bound of the bond dimension in the gathers: 4 (single-codon trains) or 8
  auto k0 = small ? ocell_kernel<0, 4> : ocell_kernel<0, 8>;
  auto k1 = small ? ocell_kernel<1, 4> : ocell_kernel<1, 8>;
  CDZ_CUDA(cudaFuncSetAttribute(k0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  CDZ_CUDA(cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  // Two internal streams forked from the caller's: sA runs the chain (PART 0 of diagonal d needs PART 0 of d+1), sB the consumers
  // (PART 1 of d needs PART 0 of d).  PART 0 of d waits for PART 1 of d+4: the pushes into the cells of diagonal d come from closing
  // cells at least four diagonals above, and the scratch / X rings are reused with that period.
  cudaStream_t sA = nullptr, sB = nullptr;
  // the chain gets the higher priority: when PART 0 of diagonal d-1 and PART 1 of diagonal d become runnable together, the CTAs of the
  // chain are placed first and the consumers fill the remaining slots
  int prio_lo = 0, prio_hi = 0;
  CDZ_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  CDZ_CUDA(cudaStreamCreateWithPriority(&sA, cudaStreamNonBlocking, prio_hi));
  CDZ_CUDA(cudaStreamCreateWithPriority(&sB, cudaStreamNonBlocking, prio_lo));
  const int mh1 = t->model->p.min_hairpin + 1;
  {
    cudaEvent_t fork;
    CDZ_CUDA(cudaEventCreateWithFlags(&fork, cudaEventDisableTiming));
    CDZ_CUDA(cudaEventRecord(fork, st));
    CDZ_CUDA(cudaStreamWaitEvent(sA, fork, 0));
    CDZ_CUDA(cudaStreamWaitEvent(sB, fork, 0));
    cudaEventDestroy(fork);
  }
  std::vector<cudaEvent_t> evB(n, nullptr);
  for (int d = n - 1; d >= 0; --d) {
    if (d + 4 <= n - 1 && evB[d + 4]) {
      CDZ_CUDA(cudaStreamWaitEvent(sA, evB[d + 4], 0));
      cudaEventDestroy(evB[d + 4]);  // (released when it has completed)
      evB[d + 4] = nullptr;
    }
    k0<<<(unsigned)(n - d), OT, smem, sA>>>(t->d_ctx, A, d, want_usage, bpp_dev);
#ifdef CDZ_EXP_NO_PART1
    if (false) {
#else
    if (d >= mh1) {
#endif
      cudaEvent_t evA;
      CDZ_CUDA(cudaEventCreateWithFlags(&evA, cudaEventDisableTiming));
      CDZ_CUDA(cudaEventRecord(evA, sA));
      CDZ_CUDA(cudaStreamWaitEvent(sB, evA, 0));
      cudaEventDestroy(evA);
#ifdef CDZ_EXP_ONE_STREAM
      k1<<<(unsigned)(n - d), OT, smem, sA>>>(t->d_ctx, A, d, want_usage, bpp_dev);
#else
      k1<<<(unsigned)(n - d), OT, smem, sB>>>(t->d_ctx, A, d, want_usage, bpp_dev);
#endif
      CDZ_CUDA(cudaEventCreateWithFlags(&evB[d], cudaEventDisableTiming));
      CDZ_CUDA(cudaEventRecord(evB[d], sB));
    }
  }
  for (cudaEvent_t e : evB)
    if (e) cudaEventDestroy(e);
  {
    cudaEvent_t ja, jb;
    CDZ_CUDA(cudaEventCreateWithFlags(&ja, cudaEventDisableTiming));
    CDZ_CUDA(cudaEventCreateWithFlags(&jb, cudaEventDisableTiming));
    CDZ_CUDA(cudaEventRecord(ja, sA));
    CDZ_CUDA(cudaEventRecord(jb, sB));
    CDZ_CUDA(cudaStreamWaitEvent(st, ja, 0));
    CDZ_CUDA(cudaStreamWaitEvent(st, jb, 0));
    cudaEventDestroy(ja);
    cudaEventDestroy(jb);
  }
  cudaStreamDestroy(sA);  // (streams with pending work are released when it has drained)
  cudaStreamDestroy(sB);
  CDZ_CUDA(cudaGetLastError());
#ifdef CDZ_OTIMING
  {
    unsigned long long h[16];
    cudaStreamSynchronize(st);
    cudaMemcpyFromSymbol(h, g_otime, sizeof(h));
    fprintf(stderr, "ocell phase cycles (sum over CTAs): gathers %llu | Qb-bar %llu | IL/IR %llu | I,G,H %llu | 4a-b %llu | 4c %llu | 4d %llu | 4e %llu | 4f %llu | usages %llu\n",
            h[0], h[1], h[2], h[3], h[4], h[5], h[6], h[7], h[8], h[9]);
    unsigned long long mx[16];
    cudaMemcpyFromSymbol(mx, g_omax, sizeof(mx));
    fprintf(stderr, "ocell phase cycles (max over CTAs):  gathers %llu | Qb-bar %llu | IL/IR %llu | I,G,H %llu | 4a-b %llu | 4c %llu | 4d %llu | 4e %llu | 4f %llu | usages %llu\n",
            mx[0], mx[1], mx[2], mx[3], mx[4], mx[5], mx[6], mx[7], mx[8], mx[9]);
    unsigned long long z[16] = {0};
    cudaMemcpyToSymbol(g_otime, z, sizeof(z));
    cudaMemcpyToSymbol(g_omax, z, sizeof(z));
  }
#endif
  return cdz_launch_usage(t, A, bpp_dev, base_dev, codon_dev, st);
}
