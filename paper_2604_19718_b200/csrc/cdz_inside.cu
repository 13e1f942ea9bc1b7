// cdz_inside.cu -- blocked wavefront inside pass (sm_100a).
//
// Every DP cell (i,j) is a small dense tensor over tensor-train bond indices and boundary nucleotides
// (eq 3.8); the recursion is DESIGN.md "Recursion".  All tables
// are row-major matrices over the packed (block-padded) bond / boundary-state index spaces,
// so the split-point sum  M2(i,j) = sum_k Qm(i,k-1) Qm1(k,j)  is the paper's flattened product
// Q_{i,k} Q_{j,k}^T (eq 3.5, Alg S4.2).
//
// Schedule: positions are grouped into blocks of <= CDZ_TB bonds; block (I,J) holds the cells whose row bond
// sigma_i lies in block I and whose column bond sigma_{j+1} lies in block J.  Block diagonals D = J-I are swept
// in order; on each one
//   1. gemm_kernel   : M2[I,J] += QM[I,K] QM1T[J,K]^T over the finished blocks I < K < J  (fp64 tensor-core
//                      mma.sync m8n8k4, cp.async pipeline, split-K partial tiles summed in fixed order),
//   2. cell_kernel   : (cdz_cell.cu) one CTA per block walks the in-block anti-diagonals, all cells of one at a time:
//                      closed cells Qb (hairpin, stack, bulge, interior <= 30, multiloop closure), Qm1 / Qml rank
//                      updates and the two in-block edge ranges of the split sum,
//   3. at D = 1,2,4,..: plan_kernel + rescale_kernel re-centre the per-position power-of-two scales (a-7).
// ext_kernel then runs the exterior recursion block column by block column.
#include <math.h>

#include <algorithm>

#include "cdz_gemm.cuh"
#include "cdz_internal.h"

namespace {

// ------------------------------------------------------------------------------------------------
// split-point GEMM: GP[I][split] = QM[I, K-range] * QM1T[J, K-range]^T, 64x64 tile per CTA, fp64 mma.sync m8n8k4
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(GEMM_THREADS) gemm_kernel(const Ctx* ctxs, int D, int nsplit) {
  extern __shared__ double gsm[];
  const Ctx& cx = ctxs[blockIdx.y];
  const int I = blockIdx.x / nsplit, sp = blockIdx.x % nsplit, J = I + D;
  if (J >= cx.tt.NB) return;
  const size_t S = (size_t)cx.tt.S;
  const int nk = D - 1;  // K blocks I+1 .. J-1
  const int kbeg = (I + 1 + (int)((long long)sp * nk / nsplit)) * CDZ_TB;
  const int kend = (I + 1 + (int)((long long)(sp + 1) * nk / nsplit)) * CDZ_TB;
  cdz_gemm_tile(cx.tab.QM + (size_t)I * CDZ_TB * S, cx.tab.QM1T + (size_t)J * CDZ_TB * S, S, kbeg, kend,
                cx.tab.GP + ((size_t)I * nsplit + sp) * (CDZ_TB * CDZ_TB), gsm);
}

// ------------------------------------------------------------------------------------------------
// CDZ_FP32_SCALED: the same contraction in single precision on the tensor cores.  Every operand row is divided by an exact power of two
// (the binary exponent of its largest finished entry, eA / eB, kept up to date by rowmax_kernel), converted to fp32 and split into two
// TF32 numbers hi + lo; a.b ~ hi.hi + hi.lo + lo.hi on mma.sync.m16n8k8.tf32 with fp32 accumulators (the dropped lo.lo term is 2^-22
// relative); the epilogue multiplies the partial tile back by 2^(eA[row] + eB[col]) in fp64 (single precision;
// line 622: rows renormalised so that the products stay in range).
// ------------------------------------------------------------------------------------------------
constexpr int CDZ_NO_EXP = -(1 << 20);
__device__ __forceinline__ unsigned f2tf32(float x) {
  unsigned r;
  asm("cvt.rna.tf32.f32 %0, %1;\n" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], const unsigned (&b)[2]) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
__device__ __forceinline__ void split_tf32(double v, double scale, unsigned& hi, unsigned& lo) {
  const float x = (float)(v * scale);
  hi = f2tf32(x);
  lo = f2tf32(x - __uint_as_float(hi));
}

__global__ void __launch_bounds__(GEMM_THREADS) gemm32_kernel(const Ctx* ctxs, int D, int nsplit) {
  extern __shared__ double gsm[];
  const Ctx& cx = ctxs[blockIdx.y];
  const int I = blockIdx.x / nsplit, sp = blockIdx.x % nsplit, J = I + D;
  if (J >= cx.tt.NB) return;
  const size_t S = (size_t)cx.tt.S;
  const int nk = D - 1;
  const int kbeg = (I + 1 + (int)((long long)sp * nk / nsplit)) * CDZ_TB;
  const int kend = (I + 1 + (int)((long long)(sp + 1) * nk / nsplit)) * CDZ_TB;
  const double* A = cx.tab.QM + (size_t)I * CDZ_TB * S;
  const double* Bm = cx.tab.QM1T + (size_t)J * CDZ_TB * S;
  double* As = gsm;
  double* Bs = gsm + GEMM_STAGES * CDZ_TB * GEMM_LD;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
  const int g = lane >> 2, tq = lane & 3;
  // exact power-of-two row scales of the fragments this thread touches
  double sa[4], sb[4];
  int ea[4], eb[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    ea[r] = max(cx.tab.eA[I * CDZ_TB + wm + r * 8 + g], -1000);  // (CDZ_NO_EXP: an all-zero row; any finite scale will do)
    eb[r] = max(cx.tab.eB[J * CDZ_TB + wn + r * 8 + g], -1000);
    sa[r] = scalbn(1.0, -ea[r]);
    sb[r] = scalbn(1.0, -eb[r]);
  }
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
  float acc[2][4][4];
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int k = 0; k < 4; ++k) acc[mi][ni][k] = 0.0f;
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
    const double* as = As + (kt % GEMM_STAGES) * CDZ_TB * GEMM_LD;
    const double* bs = Bs + (kt % GEMM_STAGES) * CDZ_TB * GEMM_LD;
#pragma unroll
    for (int k8 = 0; k8 < GEMM_BK / 8; ++k8) {
      unsigned ah[2][4], al[2][4], bh[4][2], bl[4][2];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi) {
        // a0 = (row g, k tq), a1 = (row g+8, k tq), a2 = (row g, k tq+4), a3 = (row g+8, k tq+4)
        const double* ap = as + (wm + mi * 16 + g) * GEMM_LD + k8 * 8 + tq;
        split_tf32(ap[0], sa[mi * 2], ah[mi][0], al[mi][0]);
        split_tf32(ap[8 * GEMM_LD], sa[mi * 2 + 1], ah[mi][1], al[mi][1]);
        split_tf32(ap[4], sa[mi * 2], ah[mi][2], al[mi][2]);
        split_tf32(ap[8 * GEMM_LD + 4], sa[mi * 2 + 1], ah[mi][3], al[mi][3]);
      }
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) {
        // b0 = (k tq, n g), b1 = (k tq+4, n g)
        const double* bp = bs + (wn + ni * 8 + g) * GEMM_LD + k8 * 8 + tq;
        split_tf32(bp[0], sb[ni], bh[ni][0], bl[ni][0]);
        split_tf32(bp[4], sb[ni], bh[ni][1], bl[ni][1]);
      }
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) {
          mma_tf32(acc[mi][ni], al[mi], bh[ni]);
          mma_tf32(acc[mi][ni], ah[mi], bl[ni]);
          mma_tf32(acc[mi][ni], ah[mi], bh[ni]);
        }
    }
  }
  asm volatile("cp.async.wait_group 0;\n" ::);
  double* C = cx.tab.GP + ((size_t)I * nsplit + sp) * (CDZ_TB * CDZ_TB);
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) {
      // c0 = (row g, col 2 tq), c1 = (g, 2 tq + 1), c2 = (g+8, 2 tq), c3 = (g+8, 2 tq + 1)
      const int r0 = wm + mi * 16 + g, c0 = wn + ni * 8 + 2 * tq;
      const int ec0 = max(cx.tab.eB[J * CDZ_TB + c0], -1000), ec1 = max(cx.tab.eB[J * CDZ_TB + c0 + 1], -1000);
      *reinterpret_cast<double2*>(C + r0 * CDZ_TB + c0) =
          make_double2(scalbn((double)acc[mi][ni][0], ea[mi * 2] + ec0), scalbn((double)acc[mi][ni][1], ea[mi * 2] + ec1));
      *reinterpret_cast<double2*>(C + (r0 + 8) * CDZ_TB + c0) =
          make_double2(scalbn((double)acc[mi][ni][2], ea[mi * 2 + 1] + ec0), scalbn((double)acc[mi][ni][3], ea[mi * 2 + 1] + ec1));
    }
}

// Row scales of the fp32 contraction: eA[row] / eB[row] = binary exponent of the largest entry of the QM / QM1T row over the finished
// blocks (0 for an all-zero row).  full = 0: fold in the block finished on diagonal D; full = 1 (after a rescale event, which shifts
// the entries of a row by column-dependent powers of two): recompute over all finished blocks.
__global__ void __launch_bounds__(256) rowmax_kernel(const Ctx* ctxs, int D, int full) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const int NB = t.NB, lane = threadIdx.x & 31;
  const size_t S = (size_t)t.S;
  for (int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w < 2 * t.S; w += gridDim.x * (blockDim.x >> 5)) {
    const int which = w >= t.S, row = which ? w - t.S : w, rb = row / CDZ_TB;
    // QM row of block-row I: finished column blocks I .. I+D;  QM1T row of block J: finished column blocks J-D .. J
    int c0, c1;
    if (!which) { c0 = (full ? rb : rb + D) * CDZ_TB; c1 = min(NB, rb + D + 1) * CDZ_TB; }
    else { c0 = max(0, rb - D) * CDZ_TB; c1 = (full ? rb + 1 : max(0, rb - D) + 1) * CDZ_TB; if (!full && rb - D < 0) c1 = c0; }
    const double* p = (which ? b.QM1T : b.QM) + (size_t)row * S;
    double mx = 0.0;
    for (int c = c0 + lane; c < c1; c += 32) mx = fmax(mx, fabs(p[c]));
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) {
      int* e = which ? b.eB : b.eA;
      const int ex = (mx > 0.0 && mx < 1.0e308) ? ilogb(mx) : CDZ_NO_EXP;  // CDZ_NO_EXP: no non-zero entry yet
      e[row] = (full || D == 0) ? ex : max(e[row], ex);
      if (!(mx < 1.0e308)) b.ctrl[1] = 1;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// per-position power-of-two scaling (replaces the random-vector Renormalize of PAPER.md line 622)
// ------------------------------------------------------------------------------------------------
// One CTA per design.  After block diagonal D: the longest cell of every block (I, I+D) gives a local growth
// rate (bits per position); positions take the mean rate of the windows covering them, the rounded prefix sums
// dP are added to the scale prefix P and every stored quantity over [i..j] is multiplied by 2^-(dP[j+1]-dP[i]).
__global__ void __launch_bounds__(1024) plan_kernel(const Ctx* ctxs, int D) {
  extern __shared__ double rate[];  // [NB] (NaN-free: 0 when the window holds no mass)
  __shared__ int s_maxe;
  const Ctx& cx = ctxs[blockIdx.x];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const int n = t.n, NB = t.NB, nw = NB - D;
  if (nw <= 0) {  // a shorter design of a heterogeneous batch that has already finished: nothing to rescale
    if (threadIdx.x == 0) b.ctrl[3] = 0;
    return;
  }
  const size_t S = (size_t)t.S;
  if (threadIdx.x == 0) s_maxe = 0;
  __syncthreads();
  for (int I = threadIdx.x; I < nw; I += blockDim.x) {
    const int i0 = t.blk_start[I], jj = min(t.blk_start[I + D + 1] - 1, n);
    double r = 0.0;
    if (jj > i0) {
      double mx = 0.0;
      for (int a = 0; a < t.sig[i0]; ++a)
        for (int c = 0; c < t.sig[jj]; ++c) mx = fmax(mx, b.QM[(size_t)(t.off[i0] + a) * S + t.off[jj] + c]);
      if (mx > 0.0 && mx < 1.0e308) {
        const int e = ilogb(mx);
        r = (double)e / (double)(jj - i0);
        atomicMax(&s_maxe, abs(e));
      } else if (!(mx < 1.0e308)) {
        atomicMax(&s_maxe, 2000);
      }
    }
    rate[I] = r;
  }
  __syncthreads();
  double* delta = b.R;  // scratch until the exterior phase
  for (int mpos = threadIdx.x; mpos < n; mpos += blockDim.x) {
    const int bm = t.posblk[mpos];
    const int lo = max(0, bm - D), hi = min(bm, nw - 1);
    double s = 0.0;
    for (int I = lo; I <= hi; ++I) s += rate[I];
    delta[mpos] = hi >= lo ? s / (double)(hi - lo + 1) : 0.0;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double acc = 0.0;
    int any = 0;
    b.dP[0] = 0;
    for (int mpos = 0; mpos < n; ++mpos) {
      acc += delta[mpos];
      const int v = (int)rint(acc);
      b.dP[mpos + 1] = v;
      any |= v;
    }
    b.dP[n + 1] = b.dP[n];
    b.ctrl[0] += 1;
    b.ctrl[2] = max(b.ctrl[2], s_maxe);
    if (s_maxe > 900) b.ctrl[1] = 1;
    b.ctrl[3] = any != 0;
  }
  __syncthreads();
  if (b.ctrl[3] == 0) return;
  for (int k = threadIdx.x; k <= n + 1; k += blockDim.x) b.scale[k] += b.dP[k];
  for (int k = threadIdx.x; k < t.S; k += blockDim.x) b.EB[k] = b.dP[t.bondpos[k]];
  for (int k = threadIdx.x; k < t.LS; k += blockDim.x) b.EL[k] = b.dP[t.lspos[k]];
  for (int k = threadIdx.x; k < t.RS; k += blockDim.x) b.ER[k] = b.dP[t.rspos[k] + 1];
  const int MS = t.MS;
  for (int mpos = threadIdx.x; mpos < n; mpos += blockDim.x) {
    const int e = -(b.dP[mpos + 1] - b.dP[mpos]);
    if (e == 0) continue;
    for (int z = t.opstart[mpos]; z < t.opstart[mpos + 1]; ++z) t.op_x[z] = scalbn(t.op_x[z], e);
    for (int k = 0; k < MS * MS; ++k) t.Tbar[(size_t)mpos * MS * MS + k] = scalbn(t.Tbar[(size_t)mpos * MS * MS + k], e);
  }
}

// rows of one table over the block diagonals <= D+2 (by storage location); rowsp/colsp: 0 bond space, 1 state space
__global__ void __launch_bounds__(256) rescale_kernel(const Ctx* ctxs, int which, int D) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  if (b.ctrl[3] == 0) return;
  double* tab;
  int rowsp = 0, colsp = 0, lower = 0;
  switch (which) {
    case 0: tab = b.QB; rowsp = 1; colsp = 1; break;
    case 1: tab = b.DD; rowsp = 1; colsp = 1; break;
    case 2: tab = b.D1; rowsp = 1; break;
    case 3: tab = b.D2T; rowsp = 2; lower = 1; break;
    case 4: tab = b.GI; break;
    case 5: tab = b.QBS; break;
    case 6: tab = b.QM; break;
    case 7: tab = b.QML; break;
    case 8: tab = b.M2; break;
    case 9: tab = b.EM; break;
    case 10: tab = b.EMT; lower = 1; break;
    case 11: tab = b.QBST; lower = 1; break;
    case 13: tab = b.XE; break;
    default: tab = b.QM1T; lower = 1; break;
  }
  const int nrows = rowsp == 1 ? t.LS : rowsp == 2 ? t.RS : t.S;
  const size_t ld = colsp ? (size_t)t.RS : (size_t)t.S;
  const int* Erow = rowsp == 1 ? b.EL : rowsp == 2 ? b.ER : b.EB;
  const int* Ecol = colsp ? b.ER : b.EB;
  const int n = t.n, NB = t.NB;
  for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
    // block of the row's bond position (a right state (y,c) of position q sits at bond position q+1)
    const int rb = rowsp == 1 ? t.posblk[t.lspos[row]] : rowsp == 2 ? t.posblk[t.rspos[row] + 1] : row / CDZ_TB;
    int c0, c1;
    if (lower) {
      c0 = max(0, rb - D - 2) * CDZ_TB;
      c1 = (rb + 1) * CDZ_TB;
    } else {
      const int cb = min(NB, rb + D + 3);
      if (colsp) {
        c0 = t.roff[min(n, t.blk_start[rb])];
        c1 = t.roff[min(n, t.blk_start[cb])];
      } else {
        c0 = rb * CDZ_TB;
        c1 = cb * CDZ_TB;
      }
    }
    const int er = Erow[row];
    double* p = tab + (size_t)row * ld;
    for (int c = c0 + threadIdx.x; c < c1; c += blockDim.x) {
      const int e = lower ? er - Ecol[c] : Ecol[c] - er;
      if (e != 0) p[c] = scalbn(p[c], -e);
    }
  }
}

// Interior-loop body state XS: after block diagonal D, column j (bond position j+1 in block Jc) was last advanced by
// block (Jc-D, Jc); the next block up reads the state of that block's top row i0, a quantity over
// [i0+2 .. j-2], so it is multiplied by 2^-(dP[j-1] - dP[i0+2]).
__global__ void __launch_bounds__(256) rescale_xs_kernel(const Ctx* ctxs, int D) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  if (b.ctrl[3] == 0) return;
  const int n = t.n, per = 27 * t.MS * t.MS;
  for (int j = blockIdx.x; j < n; j += gridDim.x) {
    const int Ir = t.posblk[j + 1] - D;
    if (Ir < 1) continue;  // no block above reads this column any more
    const int i0 = t.blk_start[Ir];
    if (j - 1 < i0 + 2) continue;
    const int e = b.dP[j - 1] - b.dP[i0 + 2];
    if (e == 0) continue;
    double* p = b.XS + (size_t)j * per;
    for (int k = threadIdx.x; k < per; k += blockDim.x) p[k] = scalbn(p[k], -e);
  }
}

// ------------------------------------------------------------------------------------------------
// exterior: Qext(j) = Qext(j-1) Tbar_j + sum_k Qext(k-1) Qbs(k,j); Z = sum_c Qext(n-1)[c]  (eq 3.7; App. A.3)
// ------------------------------------------------------------------------------------------------
// QX[off[k]+s] = Qext(k-1)[s].  Launch K finishes the bond positions of block K (every CTA repeats the short
// serial in-block part from a shared-memory copy of the diagonal tile of QBS) and pushes their contribution
// sum_{kb in K} QX[kb] QBS[kb, c'] into the accumulator R of every later column c'.
__global__ void __launch_bounds__(256) ext_kernel(const Ctx* ctxs, int K) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  if (K >= t.NB) return;
  __shared__ double Dg[CDZ_TB * (CDZ_TB + 1)];
  __shared__ double qx[CDZ_TB];
  const int n = t.n, MS = t.MS;
  const size_t S = (size_t)t.S;
  const int base = K * CDZ_TB;
  for (int e = threadIdx.x; e < CDZ_TB * CDZ_TB; e += blockDim.x) {
    const int r = e / CDZ_TB, c = e % CDZ_TB;
    Dg[r * (CDZ_TB + 1) + c] = b.QBS[(size_t)(base + r) * S + base + c];
  }
  // everything the serial in-block recursion reads from global memory is staged first (it is a chain of ~64 dependent steps)
  __shared__ double Rs[CDZ_TB];                                  // accumulated contributions of the earlier block rows
  __shared__ double Tbs[(CDZ_TB + CDZ_MAX_BOND) * CDZ_MAX_BOND];  // Tbar of positions p0-1 .. p1-2, compact: Sigma_pos x Sigma_{pos+1} each
  __shared__ int tof[CDZ_TB + 2];                                // their offsets in Tbs
  __shared__ double qprev[CDZ_MAX_BOND];                         // Qext of the last position of the previous block
  __shared__ int sg[CDZ_TB + 2], of[CDZ_TB + 2];                 // sigma / offset of positions p0-1 .. p1-1
  const int p0 = t.blk_start[K], p1 = min(t.blk_start[K + 1], n + 1);
  if (threadIdx.x < CDZ_TB) { qx[threadIdx.x] = 0.0; Rs[threadIdx.x] = b.R[base + threadIdx.x]; }
  for (int k = threadIdx.x; k <= p1 - p0; k += blockDim.x) {
    const int pos = p0 - 1 + k;
    sg[k] = pos >= 0 ? t.sig[pos] : 0;
    of[k] = pos >= 0 ? t.off[pos] : 0;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int acc = 0;
    for (int k = 0; k < p1 - p0; ++k) { tof[k] = acc; acc += sg[k] * sg[k + 1]; }
  }
  __syncthreads();
  for (int k = threadIdx.x / 64; k < p1 - p0; k += blockDim.x / 64) {  // 64 lanes per position
    const int pos = p0 - 1 + k, Sa = sg[k], Sc = sg[k + 1];
    for (int e = threadIdx.x % 64; e < Sa * Sc; e += 64)
      Tbs[tof[k] + e] = pos >= 0 ? t.Tbar[((size_t)pos * MS + e / Sc) * MS + e % Sc] : 0.0;
  }
  if (threadIdx.x < CDZ_MAX_BOND) qprev[threadIdx.x] = (p0 >= 1 && threadIdx.x < t.sig[p0 - 1]) ? b.Qext[t.off[p0 - 1] + threadIdx.x] : 0.0;
  __syncthreads();
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    for (int jj = p0; jj < p1; ++jj) {
      const int kk = jj - p0 + 1;  // index of position jj in sg / of; position jj-1 is kk-1
      const int Sj = sg[kk], oj = of[kk] - base;
      for (int c = 0; c < Sj; ++c) {
        double v = 0.0;
        if (jj == 0) {
          v = 1.0;
        } else {
          double part = qx[lane] * Dg[lane * (CDZ_TB + 1) + oj + c] + qx[lane + 32] * Dg[(lane + 32) * (CDZ_TB + 1) + oj + c];
          for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
          v = Rs[oj + c] + part;
          const int Sp = sg[kk - 1], op = of[kk - 1];
          const double* Tb = Tbs + tof[kk - 1];
          for (int s = 0; s < Sp; ++s) {
            const double q = op >= base ? qx[op - base + s] : qprev[s];
            v += q * Tb[s * Sj + c];
          }
        }
        __syncwarp();
        if (lane == 0) qx[oj + c] = v;
        __syncwarp();
      }
    }
  }
  __syncthreads();
  if (blockIdx.x == 0) {
    if (threadIdx.x < CDZ_TB) b.Qext[base + threadIdx.x] = qx[threadIdx.x];
    if (K == t.NB - 1 && threadIdx.x == 0) {
      double Z = 0.0;
      for (int c = 0; c < t.sig[n]; ++c) Z += qx[t.off[n] - base + c];
      const double ls = 0.6931471805599453 * (double)b.scale[n];
      b.result[0] = log(Z) + ls;
      b.result[1] = Z;
      b.result[2] = ls;
    }
  }
  for (int col = base + CDZ_TB + blockIdx.x * blockDim.x + threadIdx.x; col < t.S; col += gridDim.x * blockDim.x) {
    double acc = 0.0;
#pragma unroll 8
    for (int r = 0; r < CDZ_TB; ++r) acc += qx[r] * b.QBS[(size_t)(base + r) * S + col];
    b.R[col] += acc;
  }
}

__global__ void init_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const int n = t.n, MS = t.MS;
  const int nops = t.opstart[n];
  const int stride = gridDim.x * blockDim.x, k0 = blockIdx.x * blockDim.x + threadIdx.x;
  for (int k = k0; k <= n + 1; k += stride) { cx.tab.scale[k] = 0; cx.tab.dP[k] = 0; }
  for (int k = k0; k < 64; k += stride) cx.tab.ctrl[k] = 0;
  for (int k = k0; k < nops; k += stride) t.op_x[k] = t.op_x0[k];
  for (int k = k0; k < n * MS * MS; k += stride) t.Tbar[k] = t.Tbar0[k];
  // E(i,i-1) = identity: the diagonal of the stretch table (padding bond indices included; they are never read)
  for (int k = k0; k < t.S; k += stride) { cx.tab.EM[(size_t)k * t.S + k] = 1.0; cx.tab.EMT[(size_t)k * t.S + k] = 1.0; }
}

__global__ void zero_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.y];
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < cx.tt.S; k += gridDim.x * blockDim.x) cx.tab.R[k] = 0.0;
}

}  // namespace

int cdz_launch_inside(cdz_tables* const* ts, int B, cudaStream_t st) {
  if (B > CDZ_MAX_BATCH) {  // independent designs: chunks of CDZ_MAX_BATCH, one launch sequence each
    for (int b0 = 0; b0 < B; b0 += CDZ_MAX_BATCH) {
      const int rc = cdz_launch_inside(ts + b0, std::min(CDZ_MAX_BATCH, B - b0), st);
      if (rc != CDZ_OK) return rc;
    }
    return CDZ_OK;
  }
  int NBmax = 1, Smax = 0, nrmax = 0;
  for (int b = 0; b < B; ++b) {
    const cdz_tt* tt = ts[b]->tt;
    NBmax = std::max(NBmax, tt->NB);
    Smax = std::max(Smax, tt->S);
    nrmax = std::max(nrmax, std::max(tt->S, std::max(tt->LS, tt->RS)));
  }
  const Ctx* d_ctxs = ts[0]->d_ctx;
  if (B > 1) {
    // the handle array of the batch lives in the first handle's workspace: no allocation, no synchronisation (the copy from
    // pageable host memory is staged before cudaMemcpyAsync returns)
    std::vector<Ctx> h(B);
    for (int b = 0; b < B; ++b) h[b] = ts[b]->h;
    CDZ_CUDA(cudaMemcpyAsync(ts[0]->h.batch, h.data(), sizeof(Ctx) * B, cudaMemcpyHostToDevice, st));
    d_ctxs = ts[0]->h.batch;
  }
  cdz_cell_cfg ccfg;
  {
    const int rc = cdz_cell_config(ts, B, &ccfg);
    if (rc != CDZ_OK) return rc;
  }
  CDZ_CUDA(cudaFuncSetAttribute(gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM));
  CDZ_CUDA(cudaFuncSetAttribute(gemm32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM));
  const bool fp32 = ts[0]->precision == CDZ_FP32_SCALED;
  for (int b = 1; b < B; ++b)
    if (ts[b]->precision != ts[0]->precision) { cdz_set_error("all designs of a batch must share one precision"); return CDZ_EINVAL; }
  // accounting: launch counts always; with profiling on, one event before every launch group (class of the group
  // that follows) so that consecutive event pairs give per-class device time on this stream
  cdz_tables* T0 = ts[0];
  for (int k = 0; k < CDZ_NCLASS; ++k) if (k != 5) T0->launches[k] = 0;
  T0->ev_class.clear();
  size_t nev = 0;
  auto mark = [&](int cls, int count) {
    T0->launches[cls] += count;
    if (!T0->profile) return;
    if (nev == T0->evs.size()) { cudaEvent_t e; cudaEventCreate(&e); T0->evs.push_back(e); }
    cudaEventRecord(T0->evs[nev++], st);
    T0->ev_class.push_back(cls);
  };
  mark(4, 1);
  init_kernel<<<dim3(32, B), 256, 0, st>>>(d_ctxs);
  int nmax = 0;
  for (int b = 0; b < B; ++b) nmax = std::max(nmax, ts[b]->tt->n);
  int next_event = std::max(1, ts[0]->rescale_first);
  for (int D = 0; D < NBmax; ++D) {
    const int nblk = NBmax - D;
    const int nsplit = cdz_nsplit(NBmax, D, B);
    if (nsplit > 0) {
      mark(0, 1);
      if (fp32) gemm32_kernel<<<dim3(nblk * nsplit, B), GEMM_THREADS, GEMM_SMEM, st>>>(d_ctxs, D, nsplit);
      else gemm_kernel<<<dim3(nblk * nsplit, B), GEMM_THREADS, GEMM_SMEM, st>>>(d_ctxs, D, nsplit);
    }
    mark(1, 1);
    cdz_launch_cells(d_ctxs, B, nblk, D, nsplit, &ccfg, st);
    if (fp32 && D + 2 < NBmax) {  // (the last contraction is on diagonal NB-1 and reads the blocks finished up to NB-2)
      mark(2, 1);
      rowmax_kernel<<<dim3(148, B), 256, 0, st>>>(d_ctxs, D, 0);
    }
    if (D == next_event && D + 1 < NBmax) {
      next_event *= 2;
      mark(2, 16);
      plan_kernel<<<B, 1024, NBmax * sizeof(double), st>>>(d_ctxs, D);
      const int gx = std::min(nrmax, 148 * 8);
      for (int which = 0; which <= 13; ++which) rescale_kernel<<<dim3(gx, B), 256, 0, st>>>(d_ctxs, which, D);
      rescale_xs_kernel<<<dim3(std::min(nmax, 148 * 8), B), 256, 0, st>>>(d_ctxs, D);
      if (fp32) rowmax_kernel<<<dim3(148, B), 256, 0, st>>>(d_ctxs, D, 1);
    }
  }
  mark(3, 1 + NBmax);
  zero_kernel<<<dim3(32, B), 256, 0, st>>>(d_ctxs);
  for (int K = 0; K < NBmax; ++K) {
    const int rem = Smax - (K + 1) * CDZ_TB;
    const int gx = std::max(1, std::min(296, (rem + 255) / 256));  // one column per thread: the push part is latency-bound
    ext_kernel<<<dim3(gx, B), 256, 0, st>>>(d_ctxs, K);
  }
  mark(7, 0);  // closing event
  T0->nev_inside = T0->ev_class.size();
  CDZ_CUDA(cudaGetLastError());
  return CDZ_OK;
}
