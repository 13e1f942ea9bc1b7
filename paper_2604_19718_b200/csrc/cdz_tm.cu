// cdz_tm.cu -- the paper's OWN recursion on the CUDA path: partition function of the tensor-based free-energy model with a
// codon tensor train, summed over every coding sequence and every unpseudoknotted structure (eqs 3.5-3.8,
// Alg S4.1 / S4.2 lines 586-622).
//
//   Q_{i,j} = sum_{k in [i:j)} Q_{i,k} Q_{j,k}^T   (i < j; eq 3.5),      Q_{j,k} = chi-hat_{k,j}(Q_{k+1,j-1})   (j > k; eqs 3.6 / 3.8)
//
// over boundary points 0..n; a block Q_{i,j} is a (gamma Sigma_i) x (gamma Sigma_j) matrix, index (sigma, zeta) -> sigma * gamma + zeta
// (line 211).  The paper evaluates the first line as one TRMM per row on the GPU (eq S4.1) and chi-hat on CPU cores (line 282);
// a row-wise TRMM re-reads the whole triangle for every row (HBM-bound).  Here both lines run on the GPU as a BLOCK WAVEFRONT: the boundary
// points are grouped into blocks of <= 64 flattened indices, block diagonals D = J - I are swept in order, and on each one
//   tm_gemm_kernel   U[I,J] partial = sum_{I<K<J} U[I,K] CT[J,K]^T over the finished blocks: fp64 DMMA tiles (cdz_gemm.cuh), split-K;
//   tm_block_kernel  one CTA per block walks the in-block anti-diagonals: (A) the closed elements chi-hat of the step's cells, one warp per
//                    cell, contracted through the dense tensor-train cores in three small stages; (B) U(i,j) = GEMM partial + the two
//                    in-block edge ranges of the k-sum as dot products of contiguous rows.
// Tables: U[(i,a)][(j,b)] = Q_{i,j} (upper, identity on the diagonal blocks) and CT[(j,d)][(k,a)] = Q_{j,k} (the lower blocks as printed),
// both S x S row-major over the block-padded flattened index space, so the k-sum of a cell is a dot product of two contiguous rows.
// Scaling: every term of every Q_{i,j} contains exactly one operator of each position i..j-1, so all operator weights are multiplied by
// an exact power of two: position q by 2^-(P[q+1] - P[q]), P[q] = floor(q r), so that a stored block is the true one times 2^-(P[j] - P[i])
// (products of adjacent intervals telescope) and log Z = log Z_stored + P[n] ln 2; r = growth rate of log2 Z per position, measured by pilot
// passes over the first 60 and 600 positions.
// Readings: DESIGN.md section 17 (the same as oracle/tensor_model.py states in its header; the two share no code).
#include <math.h>

#include <algorithm>
#include <vector>

#include "cdz_gemm.cuh"
#include "cdz_internal.h"

namespace {

constexpr int TM_MAXG = 8;        // gamma
constexpr int TM_MAXXI = 4;       // xi
constexpr int TM_MAXM = 32;       // gamma * Sigma: dimension of one boundary point
constexpr int TM_THREADS = 256;
constexpr int TM_MAXCELL = 64;    // cells of one in-block anti-diagonal (a block holds <= 64 boundary points)
// shared pools of one in-block anti-diagonal.  Its cells (i, j) have i+1 in block I or the first point after it and j-1 in block J or the last
// point before it, so sum m_{i+1} <= 96, sum m_{i+1}^2 <= 32 * 96 (likewise for j-1) and by Cauchy-Schwarz sum m_{i+1} m_{j-1} <= 3072 staged X
// entries (+ <= 96 row pads); the two intermediates of chi-hat hold pairs x xi x Sigma x Sigma' entries per cell, in total
// <= pairs x xi x MS x 96 / gamma, which tm_check bounds by TM_POOL.
constexpr int TM_XPOOL = 3200, TM_POOL = 6144;
constexpr int TM_BLOCK_SMEM = (TM_XPOOL + 2 * TM_POOL) * (int)sizeof(double);

struct TmDev {
  int n, gamma, xi, mh, MS, NB, S, npair;
  int px[16], py[16];  // the nucleotide pairs with a non-zero B
  const int* sig;      // [n+1]  Sigma of every boundary point
  const int* off;      // [n+2]  padded offset of every boundary point in the flattened index space
  const int* blk;      // [NB+1] first boundary point of every block; blk[NB] = n+1
  const int* pos;      // [S]    boundary point of every flattened index (padding: the point of the block's last entry)
  const double* T;     // [n][4][MS][MS] dense tensor-train cores (operator weights summed, scaled by 2^-e)
  const double* V;     // [4][g][g]
  const double* B;     // [4][4][xi][g][g]
  const double* SB;    // [4][4][xi][g][g]   SB[y][x][rho][d][c] = sum_e S[d][e] B[y][x][rho][e][c]   (Tr_S[B X] = sum_{c,d} SB[d][c] X[c][d])
  const double* Sm;    // [g][g]
  double* U;           // S x S
  double* CT;          // S x S
  double* GP;          // split-K partial tiles [block row][split][64 x 64]
  double* result;      // [0] = Z in the stored scale
};

__global__ void tm_init_kernel(TmDev t) {
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p <= t.n; p += gridDim.x * blockDim.x)
    for (int a = 0; a < t.gamma * t.sig[p]; ++a) t.U[(size_t)(t.off[p] + a) * t.S + t.off[p] + a] = 1.0;  // Q_{i,i} = I (eq 3.6, first case)
}

__global__ void __launch_bounds__(GEMM_THREADS) tm_gemm_kernel(TmDev t, int D, int nsplit) {
  extern __shared__ double gsm[];
  const int I = blockIdx.x / nsplit, sp = blockIdx.x % nsplit, J = I + D;
  const int nk = D - 1;  // K blocks I+1 .. J-1
  const int kbeg = (I + 1 + (int)((long long)sp * nk / nsplit)) * CDZ_TB;
  const int kend = (I + 1 + (int)((long long)(sp + 1) * nk / nsplit)) * CDZ_TB;
  cdz_gemm_tile(t.U + (size_t)I * CDZ_TB * t.S, t.CT + (size_t)J * CDZ_TB * t.S, (size_t)t.S, kbeg, kend,
                t.GP + ((size_t)I * nsplit + sp) * (CDZ_TB * CDZ_TB), gsm);
}

// sum_{c,d} SB[d][c] X[c][d] for one gamma x gamma sub-block (row stride ld): compile-time gamma for the common model dimensions
template <int G>
__device__ __forceinline__ double tm_trace(const double* __restrict__ sb, const double* __restrict__ xb, int ld) {
  double v = 0.0;
#pragma unroll
  for (int cc = 0; cc < G; ++cc)
#pragma unroll
    for (int dd = 0; dd < G; ++dd) v += sb[dd * G + cc] * xb[cc * ld + dd];
  return v;
}

__global__ void __launch_bounds__(TM_THREADS) tm_block_kernel(TmDev t, int D, int nsplit) {
  // prefix sums over the cells of one in-block anti-diagonal: outputs | staged X entries | t entries | m entries | 4 x 4 output tiles
  __shared__ int pre[TM_MAXCELL + 1], prx[TM_MAXCELL + 1], prt[TM_MAXCELL + 1], prm[TM_MAXCELL + 1], prb[TM_MAXCELL + 1];
  __shared__ int overflow;
  __shared__ int boff[16 * TM_MAXXI];  // offset of B[x][y][rho] for every (pairable (x, y), rho), in the order of the intermediates
  extern __shared__ double pool[];  // X pool [TM_XPOOL] | t pool [TM_POOL] | m pool [TM_POOL]
  double* xP = pool;
  double* tP = pool + TM_XPOOL;
  double* mP = tP + TM_POOL;
  const int I = blockIdx.x, J = I + D;
  const int tid = threadIdx.x;
  const int g = t.gamma, g2 = g * g, xi = t.xi, MS = t.MS, MS2 = MS * MS, npx = t.npair * xi;
  const size_t S = (size_t)t.S;
  const int i0 = t.blk[I], i1 = t.blk[I + 1], j0 = t.blk[J], j1 = t.blk[J + 1];
  const int dmin = max(1, j0 - (i1 - 1)), dmax = (j1 - 1) - i0;
  for (int k = threadIdx.x; k < t.npair * t.xi; k += TM_THREADS) {
    const int pr = k / t.xi, rho = k - pr * t.xi;
    boff[k] = ((t.px[pr] * 4 + t.py[pr]) * t.xi + rho) * t.gamma * t.gamma;
  }
  __syncthreads();
  // item -> (cell, index inside the cell) through a prefix array
  auto cell_of = [&](const int* pr, int it, int& c) { c = 0; while (pr[c + 1] <= it) ++c; return it - pr[c]; };
  for (int d = dmin; d <= dmax; ++d) {
    const int ilo = max(i0, j0 - d), ihi = min(i1 - 1, j1 - 1 - d);
    const int ncell = ihi - ilo + 1;
    if (ncell <= 0) continue;
    const bool pairs = d >= 2 && d - 2 >= t.mh;
    if (tid == 0) {
      int ao = 0, ax = 0, at = 0, am = 0, ab = 0;
      for (int c = 0; c < ncell; ++c) {
        const int i = ilo + c, j = i + d;
        pre[c] = ao; prx[c] = ax; prt[c] = at; prm[c] = am; prb[c] = ab;
        ao += g2 * t.sig[i] * t.sig[j];
        ab += ((g * t.sig[i] + 3) >> 2) * ((g * t.sig[j] + 3) >> 2);  // 4 x 4 output tiles of phase B
        if (pairs) {
          ax += g * t.sig[i + 1] * (g * t.sig[j - 1] + 1);  // rows padded by one
          at += npx * t.sig[i + 1] * t.sig[j - 1];
          am += npx * t.sig[i] * t.sig[j];
        }
      }
      pre[ncell] = ao; prx[ncell] = ax; prt[ncell] = at; prm[ncell] = am; prb[ncell] = ab;
      // guard of the pool bounds derived above (never expected to fire): report instead of writing out of bounds
      overflow = (ncell > TM_MAXCELL || ax > TM_XPOOL || at > TM_POOL || am > TM_POOL) ? 1 : 0;
      if (overflow) t.result[1] = 1.0;
    }
    __syncthreads();
    if (overflow) return;
    // ---- (A) closed elements Q_{j,i} = chi-hat_{i,j}(Q_{i+1,j-1}) of the step's cells (eq 3.8); every stage spread over the whole CTA ----
    if (d == 1) {
      // unpaired base i:  sum_x T_i[x] (x) V[x]
      for (int it = tid; it < pre[ncell]; it += TM_THREADS) {
        int c;
        const int e = cell_of(pre, it, c), i = ilo + c, j = i + 1, mj = g * t.sig[j];
        const int al = e / mj, de = e - al * mj, sa = al / g, za = al - sa * g, sd = de / g, zd = de - sd * g;
        const double* Ti = t.T + (size_t)i * 4 * MS2;
        double v = 0.0;
#pragma unroll
        for (int x = 0; x < 4; ++x) v += Ti[x * MS2 + sa * MS + sd] * t.V[x * g2 + za * g + zd];
        t.CT[(size_t)(t.off[j] + de) * S + t.off[i] + al] = v;
      }
    } else if (pairs) {
      // base pair i.(j-1) around the block X = Q_{i+1,j-1}
      // 0: stage every X (coalesced rows) into shared memory
      for (int it = tid; it < prx[ncell]; it += TM_THREADS) {
        int c;
        const int e = cell_of(prx, it, c), i = ilo + c, l = i + d - 1, ld = g * t.sig[l] + 1;
        const int r = e / ld, cc = e - r * ld;
        if (cc < ld - 1) xP[it] = t.U[(size_t)(t.off[i + 1] + r) * S + t.off[l] + cc];
      }
      __syncthreads();
      // 1: t[pr][rho][a'][c'] = Tr_S[ B_{j,i}^rho X^{a',c'} ] = sum_{c,d} SB[y][x][rho][d][c] X[(a',c)][(c',d)]
      for (int it = tid; it < prt[ncell]; it += TM_THREADS) {
        int c;
        const int e = cell_of(prt, it, c), i = ilo + c, l = i + d - 1, s1 = t.sig[i + 1], s2 = t.sig[l], ld = g * s2 + 1;
        const int c1 = e % s2, a1 = (e / s2) % s1, rho = (e / (s1 * s2)) % xi, pr = e / (s1 * s2 * xi);
        const double* sb = t.SB + (size_t)((t.py[pr] * 4 + t.px[pr]) * xi + rho) * g2;
        const double* xb = xP + prx[c] + (a1 * g) * ld + c1 * g;
        double v = 0.0;
        if (g == 4) v = tm_trace<4>(sb, xb, ld);
        else if (g == 2) v = tm_trace<2>(sb, xb, ld);
        else if (g == 8) v = tm_trace<8>(sb, xb, ld);
        else
          for (int cc = 0; cc < g; ++cc)
            for (int dd = 0; dd < g; ++dd) v += sb[dd * g + cc] * xb[cc * ld + dd];
        tP[it] = v;
      }
      __syncthreads();
      // 2: m[pr][rho][sa][sd] = sum_{a',c'} T_i[x][sa][a'] t[pr][rho][a'][c'] T_l[y][c'][sd]
      for (int it = tid; it < prm[ncell]; it += TM_THREADS) {
        int c;
        const int e = cell_of(prm, it, c), i = ilo + c, j = i + d, l = j - 1;
        const int si = t.sig[i], sj = t.sig[j], s1 = t.sig[i + 1], s2 = t.sig[l];
        const int sd = e % sj, sa = (e / sj) % si, rho = (e / (si * sj)) % xi, pr = e / (si * sj * xi);
        const double* ti = t.T + (size_t)i * 4 * MS2 + t.px[pr] * MS2 + sa * MS;
        const double* tl = t.T + (size_t)l * 4 * MS2 + t.py[pr] * MS2 + sd;
        const double* tw = tP + prt[c] + (pr * xi + rho) * s1 * s2;
        // the two core rows are loaded once, all loads in flight together (bond dimension <= CDZ_MAX_BOND; a missing entry is 0)
        double tav[CDZ_MAX_BOND], tlv[CDZ_MAX_BOND];
#pragma unroll
        for (int u = 0; u < CDZ_MAX_BOND; ++u) {
          tav[u] = u < s1 ? ti[u] : 0.0;
          tlv[u] = u < s2 ? tl[u * MS] : 0.0;
        }
        double v = 0.0;
#pragma unroll
        for (int a1 = 0; a1 < CDZ_MAX_BOND; ++a1) {
          if (a1 < s1) {
            double sm = 0.0;
#pragma unroll
            for (int c1 = 0; c1 < CDZ_MAX_BOND; ++c1)
              if (c1 < s2) sm += tw[a1 * s2 + c1] * tlv[c1];
            v += tav[a1] * sm;
          }
        }
        mP[it] = v;
      }
      __syncthreads();
      // 3: C[(sa,za)][(sd,zd)] = sum_{pr,rho} B[x][y][rho][za][zd] m[pr][rho][sa][sd]
      for (int it = tid; it < pre[ncell]; it += TM_THREADS) {
        int c;
        const int e = cell_of(pre, it, c), i = ilo + c, j = i + d, si = t.sig[i], sj = t.sig[j], mj = g * sj;
        const int al = e / mj, de = e - al * mj, sa = al / g, za = al - sa * g, sd = de / g, zd = de - sd * g;
        const double* mw = mP + prm[c] + sa * sj + sd;
        const double* bz = t.B + za * g + zd;
        const int sij = si * sj;
        double v = 0.0;
#pragma unroll 4
        for (int k = 0; k < npx; ++k) v += bz[boff[k]] * mw[k * sij];
        t.CT[(size_t)(t.off[j] + de) * S + t.off[i] + al] = v;
      }
    }
    // spans 2 .. min_hairpin + 1 close nothing: the zero-initialised table entry stands (line 483)
    __syncthreads();
    // ---- (B) Q_{i,j} = sum_{k in [i:j)} Q_{i,k} Q_{j,k}^T: the partial tiles of the GEMM + the bonds of block I from i on + those of block J before j.
    //      4 x 4 output tiles, 8 lanes per tile striding the contiguous bond range (coalesced 64-byte row segments), butterfly over the 8 lanes ----
    {
      const int sub = tid & 7;
      const unsigned gmask = 0xFFu << (tid & 24);
      for (int tile = tid >> 3; tile < prb[ncell]; tile += TM_THREADS / 8) {
        int c;
        const int e = cell_of(prb, tile, c), i = ilo + c, j = i + d, mi = g * t.sig[i], mj = g * t.sig[j];
        const int tbn = (mj + 3) >> 2, al0 = (e / tbn) * 4, de0 = (e % tbn) * 4;
        const double* ru = t.U + (size_t)(t.off[i] + al0) * S;
        const double* rc = t.CT + (size_t)(t.off[j] + de0) * S;
        const int nr = min(4, mi - al0), nc = min(4, mj - de0);
        // rows beyond the cell (nr, nc < 4) are read from row 0 of the tile and discarded
        const size_t o1 = nr > 1 ? S : 0, o2 = nr > 2 ? 2 * S : 0, o3 = nr > 3 ? 3 * S : 0;
        const size_t p1 = nc > 1 ? S : 0, p2 = nc > 2 ? 2 * S : 0, p3 = nc > 3 ? 3 * S : 0;
        double acc[4][4];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int q = 0; q < 4; ++q) acc[r][q] = 0.0;
        auto range = [&](int lo, int hi) {
#pragma unroll 2
          for (int kb = lo + sub; kb < hi; kb += 8) {
            const double u0 = ru[kb], u1 = ru[o1 + kb], u2 = ru[o2 + kb], u3 = ru[o3 + kb];
            const double c0 = rc[kb], c1 = rc[p1 + kb], c2 = rc[p2 + kb], c3 = rc[p3 + kb];
            acc[0][0] += u0 * c0; acc[0][1] += u0 * c1; acc[0][2] += u0 * c2; acc[0][3] += u0 * c3;
            acc[1][0] += u1 * c0; acc[1][1] += u1 * c1; acc[1][2] += u1 * c2; acc[1][3] += u1 * c3;
            acc[2][0] += u2 * c0; acc[2][1] += u2 * c1; acc[2][2] += u2 * c2; acc[2][3] += u2 * c3;
            acc[3][0] += u3 * c0; acc[3][1] += u3 * c1; acc[3][2] += u3 * c2; acc[3][3] += u3 * c3;
          }
        };
        if (I == J) {
          range(t.off[i], t.off[j]);
        } else {
          range(t.off[i], (I + 1) * CDZ_TB);
          range(J * CDZ_TB, t.off[j]);
        }
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            double v = acc[r][q];
            v += __shfl_xor_sync(gmask, v, 1);
            v += __shfl_xor_sync(gmask, v, 2);
            v += __shfl_xor_sync(gmask, v, 4);
            acc[r][q] = v;
          }
        // lane `sub` finishes the two entries (r, 2 (sub & 1)) and (r, 2 (sub & 1) + 1), r = sub >> 1
        const int r = sub >> 1;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int q = 2 * (sub & 1) + h;
          double v = 0.0;
#pragma unroll
          for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int qq = 0; qq < 4; ++qq) v = (rr == r && qq == q) ? acc[rr][qq] : v;
          if (r < nr && q < nc) {
            const int ri = t.off[i] + al0 + r, rj = t.off[j] + de0 + q;
            // split-K partials: batches of 8 loads in flight before the first add (same order of the adds as a plain loop)
            const double* gp = t.GP + (size_t)I * nsplit * (CDZ_TB * CDZ_TB) + (size_t)(ri - I * CDZ_TB) * CDZ_TB + (rj - J * CDZ_TB);
            for (int s0 = 0; s0 < nsplit; s0 += 8) {
              double gv[8];
#pragma unroll
              for (int u = 0; u < 8; ++u) gv[u] = s0 + u < nsplit ? gp[(size_t)(s0 + u) * (CDZ_TB * CDZ_TB)] : 0.0;
#pragma unroll
              for (int u = 0; u < 8; ++u) v += gv[u];
            }
            t.U[(size_t)ri * S + rj] = v;
          }
        }
      }
    }
    __syncthreads();
  }
}

// Z = sum_{sigma_n} Tr_S[ Q_{0,n}^{(0, sigma_n)} ]  (eq 3.7 with the open chain of lines 561-567)
__global__ void tm_final_kernel(TmDev t) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int g = t.gamma;
  double z = 0.0;
  for (int s = 0; s < t.sig[t.n]; ++s)
    for (int d = 0; d < g; ++d)
      for (int e = 0; e < g; ++e) z += t.Sm[d * g + e] * t.U[(size_t)(t.off[0] + e) * t.S + t.off[t.n] + s * g + d];
  t.result[0] = z;
}

// ---- stochastic traceback of Q (section 4a; the alternatives of Alg S4.4, taken per sample) -------------------------
// One warp per sample; a stack of recursion elements; every decision lists its alternatives in the fixed order of DESIGN.md section 17, the
// lanes take 32 at a time with a shuffle prefix sum and stop at the first whose running sum exceeds u x (stored entry).  All weights of one
// decision carry the same power-of-two scale as the entry they decompose, so the scales never enter.
struct TmItem { int upper, i, j, a, b; };
enum { TMK_TOP = 16, TMK_UPPER = 17, TMK_UNPAIRED = 18, TMK_PAIR = 19 };

__device__ __forceinline__ uint64_t tm_mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double tm_uniform(uint64_t seed, uint64_t sample, uint64_t kind, uint64_t i, uint64_t j) {
  uint64_t h = seed;
  h = tm_mix64(h + 0x9E3779B97F4A7C15ULL * (sample + 1));
  h = tm_mix64(h + 0x9E3779B97F4A7C15ULL * (kind + 1));
  h = tm_mix64(h + 0x9E3779B97F4A7C15ULL * (i + 1));
  h = tm_mix64(h + 0x9E3779B97F4A7C15ULL * (j + 1));
  return (double)(h >> 11) * (1.0 / 9007199254740992.0);
}
// index of the first of `count` alternatives whose running sum exceeds thr; the last positive one if rounding leaves thr above all
template <typename F>
__device__ __forceinline__ int tm_pick(int lane, double thr, int count, F weight) {
  double run = 0.0;
  int last = -1;
  for (int b0 = 0; b0 < count; b0 += 32) {
    const int idx = b0 + lane;
    double w = idx < count ? weight(idx) : 0.0;
    if (!(w > 0.0)) w = 0.0;
    double sm = w;
    for (int o = 1; o < 32; o <<= 1) {
      const double v = __shfl_up_sync(0xffffffffu, sm, o);
      if (lane >= o) sm += v;
    }
    const unsigned posm = __ballot_sync(0xffffffffu, w > 0.0);
    const unsigned hit = __ballot_sync(0xffffffffu, w > 0.0 && run + sm > thr);
    if (hit) return b0 + __ffs(hit) - 1;
    if (posm) last = b0 + 31 - __clz(posm);
    run += __shfl_sync(0xffffffffu, sm, 31);
  }
  return last;
}

__global__ void __launch_bounds__(128) tm_sample_kernel(TmDev t, int J, uint64_t seed, uint8_t* seq_out, int32_t* pair_out, TmItem* stacks,
                                                        int cap) {
  const int lane = threadIdx.x & 31;
  const int smp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (smp >= J) return;
  const int n = t.n, g = t.gamma, g2 = g * g, xi = t.xi, MS = t.MS, MS2 = MS * MS;
  const size_t S = (size_t)t.S;
  uint8_t* seq = seq_out + (size_t)smp * n;
  int32_t* pair = pair_out + (size_t)smp * n;
  TmItem* stk = stacks + (size_t)smp * cap;
  for (int k = lane; k < n; k += 32) { seq[k] = 255; pair[k] = -1; }
  __syncwarp();
  int sp = 0;
  {
    // TOP: (s, d, e) ascending: S[d][e] Q_{0,n}[(0,e)][(s,d)]
    const int cnt = t.sig[n] * g2;
    auto wf = [&](int idx) {
      const int e = idx % g, d = (idx / g) % g, s = idx / g2;
      return t.Sm[d * g + e] * t.U[(size_t)(t.off[0] + e) * S + t.off[n] + s * g + d];
    };
    double tot = 0.0;
    for (int idx = lane; idx < cnt; idx += 32) { const double w = wf(idx); if (w > 0.0) tot += w; }
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    const int pick = tm_pick(lane, tm_uniform(seed, smp, TMK_TOP, 0, 0) * tot, cnt, wf);
    const int e = pick % g, d = (pick / g) % g, s = pick / g2;
    if (lane == 0) stk[0] = TmItem{1, 0, n, e, s * g + d};
    sp = 1;
    __syncwarp();
  }
  while (sp > 0) {
    --sp;
    const TmItem it = stk[sp];
    __syncwarp();
    if (it.upper) {
      const int i = it.i, j = it.j;
      if (i == j) continue;
      // UPPER(i,j,a,b): k in [i:j) ascending, c ascending = the flattened indices off[i] .. off[j]-1 (padding entries are zero and skipped)
      const double* ru = t.U + (size_t)(t.off[i] + it.a) * S;
      const double* rc = t.CT + (size_t)(t.off[j] + it.b) * S;
      const int kb0 = t.off[i], cnt = t.off[j] - kb0;
      const double thr = tm_uniform(seed, smp, TMK_UPPER, i, j) * ru[t.off[j] + it.b];
      const int pick = tm_pick(lane, thr, cnt, [&](int idx) { return ru[kb0 + idx] * rc[kb0 + idx]; });
      const int kb = kb0 + pick, k = t.pos[kb], c = kb - t.off[k];
      if (lane == 0) {
        if (k > i) stk[sp] = TmItem{1, i, k, it.a, c};
        stk[sp + (k > i ? 1 : 0)] = TmItem{0, j, k, it.b, c};
      }
      sp += k > i ? 2 : 1;
      __syncwarp();
    } else {
      const int j = it.i, k = it.j, b = it.a, c = it.b;  // LOWER(j,k,b,c): row b of point j, column c of point k
      const int sc_ = c / g, zc = c - sc_ * g, sb_ = b / g, zb = b - sb_ * g;
      const double total = t.CT[(size_t)(t.off[j] + b) * S + t.off[k] + c];
      if (j == k + 1) {
        // unpaired base k: x ascending: T_k[x][sigma(c)][sigma(b)] V[x][zeta(c)][zeta(b)]
        const double* Tk = t.T + (size_t)k * 4 * MS2;
        const int x = tm_pick(lane, tm_uniform(seed, smp, TMK_UNPAIRED, k, j) * total, 4,
                              [&](int xx) { return Tk[xx * MS2 + sc_ * MS + sb_] * t.V[xx * g2 + zc * g + zb]; });
        if (lane == 0) seq[k] = (uint8_t)x;
      } else {
        // pair k.l, l = j-1: (x, y, s1, s2, rho, cc, dd) ascending
        const int l = j - 1, s1n = t.sig[k + 1], s2n = t.sig[l];
        const double* Tk = t.T + (size_t)k * 4 * MS2;
        const double* Tl = t.T + (size_t)l * 4 * MS2;
        const double* X = t.U + (size_t)t.off[k + 1] * S + t.off[l];
        const int per = s1n * s2n * xi * g2, cnt = t.npair * per;
        auto wf = [&](int idx) {
          const int dd = idx % g, cc = (idx / g) % g, rho = (idx / g2) % xi, s2 = (idx / (g2 * xi)) % s2n, s1 = (idx / (g2 * xi * s2n)) % s1n;
          const int pr = idx / per, x = t.px[pr], y = t.py[pr];
          const double tk = Tk[x * MS2 + sc_ * MS + s1];
          if (tk == 0.0) return 0.0;
          return tk * Tl[y * MS2 + s2 * MS + sb_] * t.B[(size_t)((x * 4 + y) * xi + rho) * g2 + zc * g + zb] *
                 t.SB[(size_t)((y * 4 + x) * xi + rho) * g2 + dd * g + cc] * X[(size_t)(s1 * g + cc) * S + s2 * g + dd];
        };
        const int pick = tm_pick(lane, tm_uniform(seed, smp, TMK_PAIR, k, j) * total, cnt, wf);
        const int dd = pick % g, cc = (pick / g) % g, s2 = (pick / (g2 * xi)) % s2n, s1 = (pick / (g2 * xi * s2n)) % s1n, pr = pick / per;
        if (lane == 0) {
          seq[k] = (uint8_t)t.px[pr];
          seq[l] = (uint8_t)t.py[pr];
          pair[k] = l;
          pair[l] = k;
          stk[sp] = TmItem{1, k + 1, l, s1 * g + cc, s2 * g + dd};
        }
        ++sp;
        __syncwarp();
      }
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------------------------------------------------
struct TmLayout {
  int n = 0, NB = 0, S = 0, MS = 1, maxsplit_tiles = 0;
  std::vector<int> sig, off, blk;
  size_t o_U = 0, o_CT = 0, o_GP = 0, o_T = 0, o_V = 0, o_B = 0, o_SB = 0, o_S = 0, o_sig = 0, o_off = 0, o_blk = 0, o_pos = 0, o_res = 0, total = 0;
  std::vector<int> pos;
};

int tm_check(const cdz_tm_params* p, const cdz_tt* tt) {
  if (!p || !tt || !p->V || !p->B || !p->S) { cdz_set_error("cdz_tm: null argument"); return CDZ_EINVAL; }
  if (p->gamma < 1 || p->gamma > TM_MAXG || p->xi < 1 || p->xi > TM_MAXXI || p->min_hairpin < 0) {
    cdz_set_error("cdz_tm: need 1 <= gamma <= 8, 1 <= xi <= 4, min_hairpin >= 0");
    return CDZ_EINVAL;
  }
  if (p->gamma * tt->MS > TM_MAXM) { cdz_set_error("cdz_tm: gamma x bond dimension exceeds 32"); return CDZ_EINVAL; }
  int npair = 0;
  const int g2 = p->gamma * p->gamma;
  for (int xy = 0; xy < 16; ++xy) {
    bool nz = false;
    for (int k = 0; k < p->xi * g2; ++k) {
      const double b = p->B[(size_t)xy * p->xi * g2 + k];
      if (!std::isfinite(b) || b < 0) { cdz_set_error("cdz_tm: B must be finite and non-negative"); return CDZ_EINVAL; }
      nz = nz || b != 0.0;
    }
    npair += nz;
  }
  for (int k = 0; k < 4 * g2; ++k)
    if (!std::isfinite(p->V[k]) || p->V[k] < 0) { cdz_set_error("cdz_tm: V must be finite and non-negative"); return CDZ_EINVAL; }
  for (int k = 0; k < g2; ++k)
    if (!std::isfinite(p->S[k]) || p->S[k] < 0) { cdz_set_error("cdz_tm: S must be finite and non-negative"); return CDZ_EINVAL; }
  if ((long long)npair * p->xi * tt->MS * (96 / p->gamma) > TM_POOL) {
    cdz_set_error("cdz_tm: pairs x xi x bond x (96 / gamma) exceeds the shared pool (6144)");
    return CDZ_EINVAL;
  }
  return CDZ_OK;
}

// boundary points 0..n of the first n positions of tt, grouped greedily into blocks of <= 64 flattened indices
TmLayout tm_layout(const cdz_tm_params* p, const cdz_tt* tt, int n) {
  TmLayout L;
  L.n = n;
  L.MS = tt->MS;
  L.sig.assign(tt->sigma.begin(), tt->sigma.begin() + n + 1);
  L.off.assign(n + 2, 0);
  int b = 0, used = 0;
  L.blk.push_back(0);
  for (int q = 0; q <= n; ++q) {
    const int m = p->gamma * L.sig[q];
    if (used + m > CDZ_TB) { ++b; used = 0; L.blk.push_back(q); }
    L.off[q] = b * CDZ_TB + used;
    used += m;
  }
  L.NB = b + 1;
  L.blk.push_back(n + 1);
  L.S = L.NB * CDZ_TB;
  L.off[n + 1] = L.S;
  for (int D = 2; D < L.NB; ++D) L.maxsplit_tiles = std::max(L.maxsplit_tiles, (L.NB - D) * cdz_nsplit(L.NB, D, 1));
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += (bytes + 255) & ~size_t(255); return r; };
  const size_t g2 = (size_t)p->gamma * p->gamma;
  L.o_res = take(64);
  L.o_U = take(sizeof(double) * (size_t)L.S * L.S);
  L.o_CT = take(sizeof(double) * (size_t)L.S * L.S);
  L.o_GP = take(sizeof(double) * (size_t)std::max(1, L.maxsplit_tiles) * CDZ_TB * CDZ_TB);
  L.o_T = take(sizeof(double) * (size_t)std::max(1, n) * 4 * L.MS * L.MS);
  L.o_V = take(sizeof(double) * 4 * g2);
  L.o_B = take(sizeof(double) * 16 * p->xi * g2);
  L.o_SB = take(sizeof(double) * 16 * p->xi * g2);
  L.o_S = take(sizeof(double) * g2);
  L.o_sig = take(sizeof(int) * (n + 1));
  L.o_off = take(sizeof(int) * (n + 2));
  L.o_blk = take(sizeof(int) * (L.NB + 1));
  L.o_pos = take(sizeof(int) * (size_t)L.S);
  L.pos.assign(L.S, 0);
  for (int q = 0; q <= n; ++q)
    for (int k = L.off[q]; k < L.off[q + 1]; ++k) L.pos[k] = q;
  L.total = o;
  return L;
}

// device view of a workspace laid out by tm_layout
TmDev tm_view(const cdz_tm_params* p, const TmLayout& L, char* base) {
  const int g = p->gamma, g2 = g * g, xi = p->xi;
  TmDev t;
  t.n = L.n; t.gamma = g; t.xi = xi; t.mh = p->min_hairpin; t.MS = L.MS; t.NB = L.NB; t.S = L.S; t.npair = 0;
  for (int xy = 0; xy < 16; ++xy) {
    bool nz = false;
    for (int k = 0; k < xi * g2; ++k) nz = nz || p->B[(size_t)xy * xi * g2 + k] != 0.0;
    if (nz) { t.px[t.npair] = xy / 4; t.py[t.npair] = xy % 4; ++t.npair; }
  }
  for (int k = t.npair; k < 16; ++k) t.px[k] = t.py[k] = 0;
  t.result = (double*)(base + L.o_res);
  t.U = (double*)(base + L.o_U);
  t.CT = (double*)(base + L.o_CT);
  t.GP = (double*)(base + L.o_GP);
  t.T = (const double*)(base + L.o_T);
  t.V = (const double*)(base + L.o_V);
  t.B = (const double*)(base + L.o_B);
  t.SB = (const double*)(base + L.o_SB);
  t.Sm = (const double*)(base + L.o_S);
  t.sig = (const int*)(base + L.o_sig);
  t.off = (const int*)(base + L.o_off);
  t.blk = (const int*)(base + L.o_blk);
  t.pos = (const int*)(base + L.o_pos);
  return t;
}

inline long long tm_P(int q, double rate) { return (long long)floor((double)q * rate); }

// one pass over the first n positions, the operator weights of position q times 2^-(P[q+1] - P[q]); Z_stored to *z_out (host)
int tm_pass(const cdz_tm_params* p, const cdz_tt* tt, int n, double rate, char* base, cudaStream_t st, double* z_out, cdz_tm_info* info) {
  const TmLayout L = tm_layout(p, tt, n);
  const int g = p->gamma, g2 = g * g, xi = p->xi, MS = L.MS, MS2 = MS * MS;
  std::vector<double> T((size_t)std::max(1, n) * 4 * MS2, 0.0), SB((size_t)16 * xi * g2, 0.0);
  for (int q = 0; q < n; ++q) {
    const double sc = ldexp(1.0, -(int)(tm_P(q + 1, rate) - tm_P(q, rate)));
    for (int z = tt->opstart[q]; z < tt->opstart[q + 1]; ++z) {
      const cdz_op& o = tt->ops[z];
      T[((size_t)q * 4 + o.b) * MS2 + o.a * MS + o.c] += o.x * sc;
    }
  }
  for (int xy = 0; xy < 16; ++xy)
    for (int r = 0; r < xi; ++r)
      for (int d = 0; d < g; ++d)
        for (int c = 0; c < g; ++c) {
          double v = 0.0;
          for (int ee = 0; ee < g; ++ee) v += p->S[d * g + ee] * p->B[((size_t)xy * xi + r) * g2 + ee * g + c];
          SB[((size_t)xy * xi + r) * g2 + d * g + c] = v;
        }
  const TmDev t = tm_view(p, L, base);
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_T, T.data(), sizeof(double) * T.size(), cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_V, p->V, sizeof(double) * 4 * g2, cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_B, p->B, sizeof(double) * 16 * xi * g2, cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_SB, SB.data(), sizeof(double) * SB.size(), cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_S, p->S, sizeof(double) * g2, cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_sig, L.sig.data(), sizeof(int) * (n + 1), cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_off, L.off.data(), sizeof(int) * (n + 2), cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_blk, L.blk.data(), sizeof(int) * (L.NB + 1), cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaMemcpyAsync(base + L.o_pos, L.pos.data(), sizeof(int) * (size_t)L.S, cudaMemcpyHostToDevice, st));
  CDZ_CUDA(cudaStreamSynchronize(st));  // the staging vectors above are pageable host memory about to go out of scope
  // with info: one event before every launch group, so that consecutive pairs give the device time of the GEMMs and of the block kernels
  std::vector<cudaEvent_t> evs;
  std::vector<int> cls;  // 0 clear / init / final, 1 gemm, 2 block
  auto mark = [&](int c) {
    if (!info) return;
    cudaEvent_t ev;
    cudaEventCreate(&ev);
    cudaEventRecord(ev, st);
    evs.push_back(ev);
    cls.push_back(c);
  };
  mark(0);
  CDZ_CUDA(cudaMemsetAsync(t.result, 0, 2 * sizeof(double), st));
  CDZ_CUDA(cudaMemsetAsync(t.U, 0, sizeof(double) * (size_t)L.S * L.S, st));
  CDZ_CUDA(cudaMemsetAsync(t.CT, 0, sizeof(double) * (size_t)L.S * L.S, st));
  CDZ_CUDA(cudaFuncSetAttribute(tm_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM));
  CDZ_CUDA(cudaFuncSetAttribute(tm_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TM_BLOCK_SMEM));
  tm_init_kernel<<<32, 256, 0, st>>>(t);
  long launches = 3, gemm_launches = 0;
  double flop = 0.0;
  for (int D = 0; D < L.NB; ++D) {
    const int nblk = L.NB - D, nsplit = cdz_nsplit(L.NB, D, 1);
    if (nsplit > 0) {
      mark(1);
      tm_gemm_kernel<<<nblk * nsplit, GEMM_THREADS, GEMM_SMEM, st>>>(t, D, nsplit);
      flop += 2.0 * nblk * (double)(D - 1) * CDZ_TB * CDZ_TB * CDZ_TB;
      ++launches;
      ++gemm_launches;
    }
    mark(2);
    tm_block_kernel<<<nblk, TM_THREADS, TM_BLOCK_SMEM, st>>>(t, D, nsplit);
    ++launches;
  }
  mark(0);
  tm_final_kernel<<<1, 32, 0, st>>>(t);
  ++launches;
  mark(0);
  double res[2] = {0.0, 0.0};
  CDZ_CUDA(cudaMemcpyAsync(res, t.result, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  CDZ_CUDA(cudaStreamSynchronize(st));
  CDZ_CUDA(cudaGetLastError());
  *z_out = res[0];
  if (res[1] != 0.0) { cdz_set_error("cdz_tm_inside: internal shared-pool bound exceeded"); return CDZ_ESTATE; }
  if (info) {
    double tot = 0.0, by[3] = {0.0, 0.0, 0.0};
    for (size_t k = 0; k + 1 < evs.size(); ++k) {
      float ms = 0.f;
      CDZ_CUDA(cudaEventElapsedTime(&ms, evs[k], evs[k + 1]));
      by[cls[k]] += ms;
      tot += ms;
    }
    for (cudaEvent_t ev : evs) cudaEventDestroy(ev);
    info->device_ms = tot;
    info->gemm_ms = by[1];
    info->block_ms = by[2];
    info->gemm_launches = gemm_launches;
    info->gemm_flop = flop;
    info->launches = launches;
    info->S = L.S;
    info->NB = L.NB;
    info->scale_rate = rate;
    info->table_bytes = (double)(2 * sizeof(double)) * L.S * L.S;
  }
  return CDZ_OK;
}

constexpr int TM_PILOT = 60;

}  // namespace

extern "C" int cdz_tm_workspace_bytes(const cdz_tm_params* p, const cdz_tt* tt, size_t* bytes) {
  const int rc = tm_check(p, tt);
  if (rc != CDZ_OK) return rc;
  if (!bytes) { cdz_set_error("cdz_tm_workspace_bytes: null argument"); return CDZ_EINVAL; }
  *bytes = tm_layout(p, tt, tt->n).total;
  return CDZ_OK;
}

extern "C" int cdz_tm_inside(const cdz_tm_params* p, const cdz_tt* tt, void* workspace_dev, size_t workspace_bytes, void* stream,
                             double* logZ_host, cdz_tm_info* info) {
  int rc = tm_check(p, tt);
  if (rc != CDZ_OK) return rc;
  if (!logZ_host) { cdz_set_error("cdz_tm_inside: logZ_host is required"); return CDZ_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cdz_set_error("cdz_tm_inside: no CUDA device (the library has no CPU path)"); return CDZ_ECUDA; }
  cudaStream_t st = (cudaStream_t)stream;
  const int n = tt->n;
  const size_t need = tm_layout(p, tt, n).total;
  char* base = (char*)workspace_dev;
  bool own = false;
  if (!base) {
    if (cudaMalloc((void**)&base, need) != cudaSuccess) { cudaGetLastError(); cdz_set_error("cdz_tm_inside: device allocation failed"); return CDZ_ENOMEM; }
    own = true;
  } else if (workspace_bytes < need) {
    cdz_set_error("cdz_tm_inside: workspace too small (cdz_tm_workspace_bytes)");
    return CDZ_EINVAL;
  }
  // pilot passes over prefixes: the growth rate of log2 Z per position (the second pilot, run with the rate of the first, pins it to
  // ~1e-2 bits per position, i.e. well inside the fp64 exponent range at 15000 nt)
  double rate = 0.0, z = 0.0;
  for (int np : {TM_PILOT, 10 * TM_PILOT}) {
    if (rc != CDZ_OK || n <= np) break;
    rc = tm_pass(p, tt, np, rate, base, st, &z, nullptr);
    if (rc == CDZ_OK && (!(z > 0.0) || !std::isfinite(z))) { cdz_set_error("cdz_tm_inside: pilot pass left the fp64 range"); rc = CDZ_EOVERFLOW; }
    if (rc == CDZ_OK) rate = (log2(z) + (double)tm_P(np, rate)) / np;
  }
  if (rc == CDZ_OK) rc = tm_pass(p, tt, n, rate, base, st, &z, info);
  if (rc == CDZ_OK && (!(z > 0.0) || !std::isfinite(z))) { cdz_set_error("cdz_tm_inside: partition function left the fp64 range"); rc = CDZ_EOVERFLOW; }
  if (rc == CDZ_OK) *logZ_host = log(z) + (double)tm_P(n, rate) * M_LN2;
  if (own) cudaFree(base);
  return rc;
}

// parity access after cdz_tm_inside with a caller workspace: which = 0 the upper block Q_{i,j} (i <= j) as [gamma Sigma_i][gamma Sigma_j],
// which = 1 the lower block Q_{j,i} (j > i) as [gamma Sigma_j][gamma Sigma_i]; true value = stored * 2^shift
extern "C" int cdz_tm_block(const cdz_tm_params* p, const cdz_tt* tt, const void* workspace_dev, double scale_rate, int which, int i,
                            int j, double* out_host, int* shift_out) {
  const int rc = tm_check(p, tt);
  if (rc != CDZ_OK) return rc;
  const int n = tt->n;
  if (!workspace_dev || !out_host || i < 0 || j < i || j > n || (which != 0 && which != 1) || (which == 1 && i == j)) {
    cdz_set_error("cdz_tm_block: bad argument");
    return CDZ_EINVAL;
  }
  const TmLayout L = tm_layout(p, tt, n);
  const char* base = (const char*)workspace_dev;
  const int mi = p->gamma * L.sig[i], mj = p->gamma * L.sig[j];
  if (which == 0) {
    CDZ_CUDA(cudaMemcpy2D(out_host, sizeof(double) * mj, base + L.o_U + sizeof(double) * ((size_t)L.off[i] * L.S + L.off[j]),
                          sizeof(double) * L.S, sizeof(double) * mj, mi, cudaMemcpyDeviceToHost));
  } else {
    CDZ_CUDA(cudaMemcpy2D(out_host, sizeof(double) * mi, base + L.o_CT + sizeof(double) * ((size_t)L.off[j] * L.S + L.off[i]),
                          sizeof(double) * L.S, sizeof(double) * mi, mj, cudaMemcpyDeviceToHost));
  }
  if (shift_out) *shift_out = (int)(tm_P(j, scale_rate) - tm_P(i, scale_rate));
  return which == 0 ? mi * mj : mj * mi;
}

extern "C" int cdz_tm_sample(const cdz_tm_params* p, const cdz_tt* tt, void* workspace_dev, int J, uint64_t seed, uint8_t* seq_dev,
                             int32_t* pair_dev, void* stream) {
  const int rc = tm_check(p, tt);
  if (rc != CDZ_OK) return rc;
  if (!workspace_dev || J < 0 || !seq_dev || !pair_dev) { cdz_set_error("cdz_tm_sample: bad argument"); return CDZ_EINVAL; }
  if (J == 0) return CDZ_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const TmLayout L = tm_layout(p, tt, tt->n);
  const TmDev t = tm_view(p, L, (char*)workspace_dev);
  // every element on the stack covers an interval disjoint from the others: at most n + 2 items
  const int cap = tt->n + 2;
  TmItem* stacks = nullptr;
  if (cudaMallocAsync((void**)&stacks, sizeof(TmItem) * (size_t)J * cap, st) != cudaSuccess) {
    cudaGetLastError();
    cdz_set_error("cdz_tm_sample: device allocation of the traceback stacks failed");
    return CDZ_ENOMEM;
  }
  tm_sample_kernel<<<(J + 3) / 4, 128, 0, st>>>(t, J, seed, seq_dev, pair_dev, stacks, cap);
  CDZ_CUDA(cudaGetLastError());
  CDZ_CUDA(cudaFreeAsync(stacks, st));
  return CDZ_OK;
}
