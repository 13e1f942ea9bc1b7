// cdz_cell.cu -- the per-cell part of the blocked wavefront inside pass (sm_100a): closed cells Qb (hairpin, stack,
// bulge, interior <= 30, multiloop closure), Qbs / Qm1 / Qml, the in-block edge ranges of the split-point sum, Qm, and
// the mismatch-dressed extensions that later interior loops read (
// sequence sums as in chi-hat, eq 3.8).
//
// One CTA (512 threads) per block (I, J = I + D).  The in-block anti-diagonals are walked in order; on each one ALL cells are
// advanced together in a few phases separated by __syncthreads:
//   P1  everything that depends only on finished diagonals; the work is handed out dynamically (shared counters), in this order:
//         X   one warp per cell: interior-loop bodies X_u (row recursion, state of every column in shared memory) and
//             XE = sum_u win[u] X_u + hairpin
//         row items, GL = 4 lanes each over a contiguous bond range: M2 edge ranges, Bl / Br (multiloop closure + bulges >= 2),
//             Z1 / Z2 (l1 = 1 / l2 = 1 interior loops)
//         single-lane items: SB (stack, bulge 1), the recursive parts of Qm1 / Qml, E(i,j)
//   P2  Y   = everything that carries the closing mismatch
//   P3  Qb  (inner[x,y;a',c'] expanded in place from Bl, Br, SB and Y)
//   P4  Qbs, Qm1, Qml, M2, Qm (+ transposed copies)  and  DD = dressed extension of Qb(i,j) over [i-1..j+1]
//   P5  GI, D1, D2T (DD summed over one or both nucleotides)
// Every band sum is a dot product of two CONTIGUOUS row segments of row-major tables (transposed copies EMT, QBST,
// D2T, QM1T exist for that purpose), so the loads of the lanes of a group are coalesced and independent.
// Position metadata, the boundary states of every window position packed 4 bits each (PosPk: the serial loops of SB / Qb / P4 / P5 extract a
// state's bond or nucleotide with a register shift instead of a dependent load) and the dense cores TL_i[(a,x)][c], TR_j[a][(y,c)] of the
// block's rows / columns live in shared memory; the per-cell intermediates live in a shared-memory scratch slab.
#include <math.h>

#include <algorithm>

#include "cdz_internal.h"

namespace {

struct PosMeta { int off, sig, loff, nL, roff, nR, ops, nuc; };  // 32 bytes per position of a window; nuc = bit mask of the nucleotides possible there

// boundary states of one position packed 4 bits each (|L_i|, |R_j| <= 16; bonds < 8, nucleotides < 4): left states (a, x) in lsa / lsx, right states
// (y, c) in rsy / rsc.  Entry k = (word >> 4 k) & 15: a register shift instead of a dependent global load in the serial loops of P1-P5.
struct PosPk { unsigned long long lsa, lsx, rsy, rsc; };
__device__ __forceinline__ int pk(unsigned long long w, int k) { return (int)(w >> (4 * k)) & 15; }

// window of position records in shared memory; -DCDZ_CHECK (development) traps on an index outside the window
struct MetaWin {
  PosMeta* p;
  int n, tag;
  __device__ __forceinline__ PosMeta& operator[](int k) const {
#ifdef CDZ_CHECK
    if (k < 0 || k >= n) {
      printf("cdz: position window %d: index %d outside [0,%d) (block %d,%d thread %d)\n", tag, k, n, blockIdx.x, blockIdx.y, threadIdx.x);
      __trap();
    }
#endif
    return p[k];
  }
};

constexpr int XU = 27;       // interior totals u = l1 + l2 = 4..30 with l1, l2 >= 2
constexpr int ROWPAD = 34;   // row window  [i0-1, i1+ROWPAD-2]
constexpr int COLPAD = 34;   // column window [j0-COLPAD+1, j1+1]

struct Dims {
  int M, ML, MR, nps;  // bond / left-state / right-state / pair-slot dimensions (strides of the scratch arrays)
  int lgM, lgR, lgP;   // ceil log2 of M, MR, nps (item decoding)
  int pc;              // percell(), filled by the host
  __host__ __device__ int percell() const { return 6 * M * M + ML * M + M * MR + 2 * ML * MR + nps * M * M; }
};

__host__ __device__ inline int clog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

struct Scr {  // scratch of one cell
  double *XE, *Bl, *Br, *Z1, *Z2, *Y, *SB, *QBc, *M2s, *R1, *R2;
};
__device__ __forceinline__ Scr scr_of(double* base, const Dims& D, int ci) {
  double* s = base + ci * D.pc;
  Scr k;
  const int MM = D.M * D.M;
  k.XE = s; s += MM;
  k.Bl = s; s += MM;
  k.Br = s; s += MM;
  k.M2s = s; s += MM;
  k.R1 = s; s += MM;
  k.R2 = s; s += MM;
  k.Z1 = s; s += D.ML * D.M;
  k.Z2 = s; s += D.M * D.MR;
  k.Y = s; s += D.ML * D.MR;
  k.QBc = s; s += D.ML * D.MR;
  k.SB = s;
  return k;
}

// shared-memory plan (bytes), identical on host and device
struct Plan {
  int nrow, ncol;        // window lengths (positions)
  int maxbond, maxls;    // compact row lists (bonds / left states of the row window)
  int ntl, ntr;          // positions with a dense TL / TR core
  size_t o_rowm, o_colm, o_rowpk, o_colpk, o_crow, o_rbpos, o_rlpos, o_rbp, o_cbp, o_tl, o_tr, o_xoff, o_xst, o_scr, total;
};
// span: largest extent, in global (block-padded) bond indices, of a row / column window
__host__ __device__ inline Plan make_plan(int maxpos, int span, const Dims& D, int C) {
  Plan p;
  p.nrow = maxpos + ROWPAD;
  p.ncol = maxpos + COLPAD + 2;
  p.maxbond = p.nrow * D.M;
  p.maxls = p.nrow * D.ML;
  p.ntl = maxpos + 2;
  p.ntr = maxpos + 3;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += (bytes + 15) & ~size_t(15); return r; };
  p.o_rowm = take(sizeof(PosMeta) * p.nrow);
  p.o_colm = take(sizeof(PosMeta) * p.ncol);
  p.o_rowpk = take(sizeof(PosPk) * p.nrow);
  p.o_colpk = take(sizeof(PosPk) * p.ncol);
  p.o_crow = take(sizeof(int) * (p.nrow + 1));
  p.o_rbpos = take(sizeof(short) * p.maxbond);
  p.o_rlpos = take(sizeof(short) * p.maxls);
  p.o_rbp = take(span);
  p.o_cbp = take(span);
  p.o_tl = take(sizeof(double) * (size_t)p.ntl * D.ML * D.M);
  p.o_tr = take(sizeof(double) * (size_t)p.ntr * D.M * D.MR);
  p.o_xoff = take(sizeof(int) * (maxpos + 2));
  p.o_xst = take(sizeof(double) * (size_t)XU * D.M * (CDZ_TB + 2 * D.M));  // X_u state of every column: 27 x M x Sigma_{j-1}
  p.o_scr = take(sizeof(double) * (size_t)C * D.percell());
  p.total = o;
  return p;
}

}  // namespace

namespace {

// One warp advances the interior-loop bodies of one cell:  X_u(i,j) = Tbar_{i+2} X_{u-1}(i+1,j) + GI(i+3, j+1-u) E(j+3-u, j-2)
// for u = 4..30 (lane = u - 4), in place in the shared-memory state xs of column j (layout [u][a2 < M][c2 < Sc]), and
// XE[a2][c2] = sum_u win[u] X_u + hairpin.  Columns are processed W at a time so that every lane keeps MA x W accumulators;
// all lanes finish reading X_{u-1} before any lane writes X_u.
template <int MA, int W>
__device__ __forceinline__ void x_cell(int lane, double* xs, int Mst, int Sa, int Sa3, int Sc, bool hasold, bool closed, int mh1,
                                       int maxint, int i, int j, const double* Tb, int MS, const double* gi, const double* em,
                                       size_t S, const PosMeta* colm, int cbase, const double* win, double hpw,
                                       const double* emh, double* xe_out, int Mxe, double* xe_glob) {
  const int u = 4 + lane;
  const bool live = lane < XU;
  const int cp = j + 3 - u;
  const bool hasnew = live && cp - (i + 2) - 3 >= mh1;
  int cpo = 0, cps = 0;
  if (hasnew) { const PosMeta mc = colm[cp - cbase]; cpo = mc.off; cps = mc.sig; }
  const double wu = (live && u <= maxint) ? win[u] : 0.0;
  for (int cc = 0; cc < Sc; cc += W) {
    const int ncw = min(W, Sc - cc);
    double acc[MA][W];
#pragma unroll
    for (int a = 0; a < MA; ++a)
#pragma unroll
      for (int w = 0; w < W; ++w) acc[a][w] = 0.0;
    // the hairpin entry this lane adds at the end of the pass (even lanes own one entry each): with a single pass per cell (bond dimension
    // <= 4) it is loaded now and used last; with several passes the early load costs more than it hides (measured)
    double ehp = 0.0;
    if (MA == 4 && (lane & 1) == 0) {
      const int e = lane >> 1, a = e / W, w = e % W;
      if (closed && a < Sa && w < ncw) ehp = emh[(size_t)a * S + cc + w];
    }
    if (live && hasold && u > 4) {
      const double* xo = xs + (size_t)(u - 5) * Mst * Sc + cc;
#pragma unroll
      for (int a3 = 0; a3 < MA; ++a3) {  // fixed trip count + predicates: all loads of the pass can be issued before the first FMA
        if (a3 < Sa3) {
          double xv[W];
#pragma unroll
          for (int w = 0; w < W; ++w) xv[w] = w < ncw ? xo[a3 * Sc + w] : 0.0;
#pragma unroll
          for (int a = 0; a < MA; ++a) {
            if (a < Sa) {
              const double tb = Tb[a * MS + a3];
#pragma unroll
              for (int w = 0; w < W; ++w) acc[a][w] += tb * xv[w];
            }
          }
        }
      }
    }
#pragma unroll
    for (int u2 = 0; u2 < MA; ++u2) {
      if (u2 >= cps) break;
      double ev[W];
#pragma unroll
      for (int w = 0; w < W; ++w) ev[w] = w < ncw ? em[(size_t)(cc + w) * S + cpo + u2] : 0.0;
#pragma unroll
      for (int a = 0; a < MA; ++a) {
        if (a < Sa) {
          const double gv = gi[(size_t)a * S + cpo + u2];
#pragma unroll
          for (int w = 0; w < W; ++w) acc[a][w] += gv * ev[w];
        }
      }
    }
    __syncwarp();
    if (live) {
      double* xn = xs + (size_t)(u - 4) * Mst * Sc + cc;
#pragma unroll
      for (int a = 0; a < MA; ++a)
        if (a < Sa)
#pragma unroll
          for (int w = 0; w < W; ++w)
            if (w < ncw) xn[a * Sc + w] = acc[a][w];
    }
    // XE: weighted sum over the lanes; MA*W (= 16) values are reduced together, halving the value set at every shuffle step
    static_assert(MA * W == 16, "transpose-reduce below assumes 16 values per lane");
    double v[16];
#pragma unroll
    for (int a = 0; a < MA; ++a)
#pragma unroll
      for (int w = 0; w < W; ++w) v[a * W + w] = wu * acc[a][w];
#pragma unroll
    for (int half = 8, bit = 16; half >= 1; half >>= 1, bit >>= 1) {
      const bool up = (lane & bit) != 0;
#pragma unroll
      for (int k = 0; k < half; ++k) {
        const double send = up ? v[k] : v[k + half];
        const double keep = up ? v[k + half] : v[k];
        v[k] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
      }
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
    if ((lane & 1) == 0) {
      const int e = lane >> 1, a = e / W, w = e % W;
      if (a < Sa && w < ncw) {
        const double xv = v[0] + (MA == 4 ? hpw * ehp : closed ? hpw * emh[(size_t)a * S + cc + w] : 0.0);
        xe_out[a * Mxe + cc + w] = xv;
        xe_glob[(size_t)a * S + cc + w] = xv;  // same index as emh: row (i+2, a), column (j-1, c)
      }
    }
    __syncwarp();
  }
}

constexpr int CELL_THREADS = 512;
constexpr int LG = 2, GL = 1 << LG;  // lanes that share one row item of the cooperative P1 loop

struct KArgs {
  int D, nsplit, C, maxpos, span;
  Dims dm;
};

// FIX = 1: the dimensions of the single-codon tensor train of cdz_tt_build (bond dimension 4, 4 left / 6 right boundary states, 6 pair slots) as
// compile-time constants, so that the small loops unroll and the item decoding folds; FIX = 0: run-time dimensions.
template <int FIX>
__global__ void __launch_bounds__(CELL_THREADS, 1) cell_kernel(const Ctx* ctxs, KArgs ka) {
  extern __shared__ __align__(16) unsigned char smraw[];
  __shared__ CModel cm;
  __shared__ int pmx[16];  // nucleotide mask of position i -> mask of the nucleotides at j that can pair with one of them
  __shared__ int p1ctr[4];  // work counters of P1: warps take X cells / 32-slot chunks of the item loops as they become free
  __shared__ double wsl[6][16];  // stack factor by (closing pair type, inner pair slot): wst[P][ptype(slot)]
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const int I = blockIdx.x, J = I + ka.D;
  if (J >= t.NB) return;
  Dims dm = ka.dm;
  if (FIX) { dm.M = 4; dm.ML = 4; dm.MR = 6; dm.nps = 6; dm.lgM = 2; dm.lgR = 3; dm.lgP = 3; dm.pc = dm.percell(); }
  const Plan pl = make_plan(ka.maxpos, ka.span, dm, ka.C);
  MetaWin rowm{(PosMeta*)(smraw + pl.o_rowm), 0, 0};
  MetaWin colm{(PosMeta*)(smraw + pl.o_colm), 0, 1};
  PosPk* rowpk = (PosPk*)(smraw + pl.o_rowpk);
  PosPk* colpk = (PosPk*)(smraw + pl.o_colpk);
  int* crow = (int*)(smraw + pl.o_crow);
  short* rbpos = (short*)(smraw + pl.o_rbpos);
  short* rlpos = (short*)(smraw + pl.o_rlpos);
  uint8_t* rbp = smraw + pl.o_rbp;  // bond index -> position (relative to the window base), row / column window
  uint8_t* cbp = smraw + pl.o_cbp;
  double* TLs = (double*)(smraw + pl.o_tl);
  double* TRs = (double*)(smraw + pl.o_tr);
  int* xoff = (int*)(smraw + pl.o_xoff);      // start of column j's X state in xst (units of M doubles per u)
  double* xst = (double*)(smraw + pl.o_xst);  // X_u(i+1, j) of every column of the block, u = 4..30
  double* scrb = (double*)(smraw + pl.o_scr);
  const int tid = threadIdx.x, NT = blockDim.x;
  const int n = t.n, MS = t.MS, MS2 = MS * MS;
  const size_t S = (size_t)t.S, RS = (size_t)t.RS;
  const int M = dm.M, ML = dm.ML, MR = dm.MR, nps = dm.nps;
  const int lgM = dm.lgM, lgR = dm.lgR;
  const int Mp = 1 << lgM, MRp = 1 << lgR;

  // rows i in [i0,i1), columns j in [j0,j1): bond position j+1 lies in block J
  const int i0 = t.blk_start[I], i1 = min(t.blk_start[I + 1], n);
  const int j0 = max(t.blk_start[J], 1) - 1, j1 = t.blk_start[J + 1] - 1;
  const int rbase = max(i0 - 1, 0), rend = min(i1 + ROWPAD - 2, n);
  const int cbase = max(j0 - COLPAD + 1, 0), cend = min(j1 + 1, n);
  const int nrp = rend - rbase + 1, ncp = cend - cbase + 1;
  rowm.n = nrp;
  colm.n = ncp;
  const int tlbase = rbase, ntl = min(i1, n - 1) - tlbase + 1;
  const int trbase = max(j0 - 1, 0), ntr = min(j1, n - 1) - trbase + 1;

  // ---- stage the model, the position metadata and the dense cores ----------------------------------------------
  {
    const int* src = (const int*)cx.cm;
    int* dst = (int*)&cm;
    for (int k = tid; k < (int)(sizeof(CModel) / 4); k += NT) dst[k] = src[k];
  }
  auto load_meta = [&](int p) {
    PosMeta m;
    m.off = t.off[p];
    m.sig = t.sig[p];
    if (p < n) {
      m.loff = t.loff[p]; m.nL = t.loff[p + 1] - m.loff;
      m.roff = t.roff[p]; m.nR = t.roff[p + 1] - m.roff;
      m.ops = t.opstart[p];
      m.nuc = 0;
      for (int l = 0; l < m.nL; ++l) m.nuc |= 1 << t.ls_x[m.loff + l];
    } else {
      m.loff = t.loff[n]; m.nL = 0; m.roff = t.roff[n]; m.nR = 0; m.ops = t.opstart[n]; m.nuc = 0;
    }
    return m;
  };
  auto load_pk = [&](int p) {
    PosPk w{0ull, 0ull, 0ull, 0ull};
    if (p < n) {
      const int l0 = t.loff[p], nl = t.loff[p + 1] - l0, r0 = t.roff[p], nr = t.roff[p + 1] - r0;
      for (int l = 0; l < nl; ++l) {
        w.lsa |= (unsigned long long)t.ls_a[l0 + l] << (4 * l);
        w.lsx |= (unsigned long long)t.ls_x[l0 + l] << (4 * l);
      }
      for (int r = 0; r < nr; ++r) {
        w.rsy |= (unsigned long long)t.rs_y[r0 + r] << (4 * r);
        w.rsc |= (unsigned long long)t.rs_c[r0 + r] << (4 * r);
      }
    }
    return w;
  };
  for (int k = tid; k < nrp; k += NT) rowm[k] = load_meta(rbase + k);
  for (int k = tid; k < ncp; k += NT) colm[k] = load_meta(cbase + k);
  // (the threads at the other end of the CTA take the packed descriptors, so that both run concurrently)
  for (int k = NT - 1 - tid; k < nrp; k += NT) rowpk[k] = load_pk(rbase + k);
  for (int k = NT - 1 - tid; k < ncp; k += NT) colpk[k] = load_pk(cbase + k);
  const int rkb0 = t.off[rbase], rkb1 = t.off[rend] + t.sig[rend];
  const int ckb0 = t.off[cbase], ckb1 = t.off[cend] + t.sig[cend];
  for (int k = tid; k < rkb1 - rkb0; k += NT) rbp[k] = (uint8_t)min(t.bondpos[rkb0 + k] - rbase, 255);
  for (int k = tid; k < ckb1 - ckb0; k += NT) cbp[k] = (uint8_t)min(t.bondpos[ckb0 + k] - cbase, 255);
  for (int k = tid; k < ntl * ML * M; k += NT) TLs[k] = 0.0;
  for (int k = tid; k < ntr * M * MR; k += NT) TRs[k] = 0.0;
  __syncthreads();
  if (tid < 16) {
    int pm = 0;
    for (int x = 0; x < 4; ++x)
      if (tid >> x & 1)
        for (int y = 0; y < 4; ++y)
          if (cm.pslot[x * 4 + y] >= 0) pm |= 1 << y;
    pmx[tid] = pm;
  }
  if (tid >= 32 && tid < 32 + 96) {
    const int P = (tid - 32) >> 4, s2 = (tid - 32) & 15;
    wsl[P][s2] = s2 < cm.nps ? cm.wst[P][cm.ptype[cm.slot_x[s2] * 4 + cm.slot_y[s2]]] : 0.0;
  }
  if (tid == 0) {
    p1ctr[0] = p1ctr[1] = p1ctr[2] = 0;
    int acc = 0;
    for (int k = 0; k < nrp; ++k) { crow[k] = acc; acc += rowm[k].sig; }
    crow[nrp] = acc;
  }
  __syncthreads();
  const int L0 = rowm[0].loff;
  for (int k = tid; k < nrp; k += NT) {
    const PosMeta m = rowm[k];
    for (int a = 0; a < m.sig; ++a) rbpos[crow[k] + a] = (short)k;
    for (int l = 0; l < m.nL; ++l) rlpos[m.loff - L0 + l] = (short)k;
  }
  for (int k = tid; k < ntl; k += NT) {
    const int p = tlbase + k;
    if (p < n)
      for (int z = t.opstart[p]; z < t.opstart[p + 1]; ++z) TLs[(k * ML + t.op_l[z]) * M + t.op_c[z]] += t.op_x[z];
  }
  for (int k = tid; k < ntr; k += NT) {
    const int p = trbase + k;
    if (p < n)
      for (int z = t.opstart[p]; z < t.opstart[p + 1]; ++z) TRs[(k * M + t.op_a[z]) * MR + t.op_r[z]] += t.op_x[z];
  }
  __syncthreads();

  // ---- interior-loop body state of the block's columns: X_u(i1, j) comes from the block below (global XS), zero on the diagonal ----
  const int ncolj = j1 - j0;
  if (tid == 0) {
    int acc = 0;
    for (int jc = 0; jc < ncolj; ++jc) { xoff[jc] = acc; acc += (j0 + jc >= 1) ? colm[j0 + jc - 1 - cbase].sig : 0; }
    xoff[ncolj] = acc;
  }
  __syncthreads();
  for (int jc = 0; jc < ncolj; ++jc) {
    const int j = j0 + jc, Sc = xoff[jc + 1] - xoff[jc];
    double* xs = xst + (size_t)XU * M * xoff[jc];
    const double* src = b.XS + (size_t)j * (XU * MS2);
    for (int e = tid; e < XU * MS * Sc; e += NT) {
      const int c2 = e % Sc, a2 = (e / Sc) % MS, u4 = e / (Sc * MS);
      xs[((size_t)u4 * M + a2) * Sc + c2] = (I != J) ? src[u4 * MS2 + a2 * MS + c2] : 0.0;
    }
  }
  __syncthreads();

  const int mh1 = cm.min_hairpin + 1, maxint = cm.max_interior;
  const double* __restrict__ Tbar = t.Tbar;

  // compact row ranges of the bond rows / left-state rows of positions [lo, hi] of the row window
  auto bond_rows = [&](int lo, int hi, int& r0) {
    lo = max(lo, rbase); hi = min(hi, rend);
    if (hi < lo) { r0 = 0; return 0; }
    r0 = crow[lo - rbase];
    return crow[hi + 1 - rbase] - r0;
  };
  auto ls_rows = [&](int lo, int hi, int& r0) {
    lo = max(lo, rbase); hi = min(hi, min(rend, n - 1));
    if (hi < lo) { r0 = 0; return 0; }
    r0 = rowm[lo - rbase].loff - L0;
    return rowm[hi - rbase].loff + rowm[hi - rbase].nL - L0 - r0;
  };

#ifdef CDZ_PHASE_TIMING
  long long tph[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tlast = clock64();
  long long ttyp[6] = {0, 0, 0, 0, 0, 0};
#define CDZ_TICK(k) do { const long long now__ = clock64(); tph[k] += now__ - tlast; tlast = now__; } while (0)
#else
#define CDZ_TICK(k)
#endif
  // dynamic distribution of the P1 work: lane 0 takes the next unit, the warp follows
  auto grab = [&](int* c) {
    int w = 0;
    if ((tid & 31) == 0) w = atomicAdd(c, 1);
    return __shfl_sync(0xffffffffu, w, 0);
  };
  const int dmin = max(0, j0 - (i1 - 1)), dmax = (j1 - 1) - i0;
  for (int d = dmin; d <= dmax; ++d) {
    const int ilo = max(i0, j0 - d), ihi = min(i1 - 1, j1 - 1 - d);
    const bool closed = d >= mh1;
    for (int clo = ilo; clo <= ihi; clo += ka.C) {
      const int chi = min(ihi, clo + ka.C - 1);
      // ================= P1: everything that reads finished diagonals only =======================================
      int rb0, rb1, rb2, rl1;
      const int nb0 = bond_rows(clo, chi, rb0);          // bonds of position i
      const int nb1 = bond_rows(clo + 1, chi + 1, rb1);  // bonds of position p = i+1
      const int nb2 = bond_rows(clo + 2, chi + 2, rb2);  // bonds of position i+2
      const int nl1 = ls_rows(clo + 1, chi + 1, rl1);    // left states of position p
      // ---- X_u / XE: one warp per cell, state of column j in shared memory ------------------------------------------------------
      if (d >= 4) {
        const int lane = tid & 31;
        for (int w; (w = grab(&p1ctr[0])) <= chi - clo;) {
          const int i = clo + w, j = i + d, kp2 = i + 2 - rbase;
          const PosMeta mq = colm[j - 1 - cbase];
          double* xs = xst + (size_t)XU * M * xoff[j - j0];
          const double* Tb = Tbar + (size_t)(i + 2) * MS2;
          const double* gi = b.GI + (size_t)rowm[kp2].off * S;
          const double* em = b.EMT + (size_t)mq.off * S;
          const double* emh = b.EM + (size_t)rowm[kp2].off * S + mq.off;
          double* xeg = b.XE + (size_t)rowm[kp2].off * S + mq.off;
          double* xe = scr_of(scrb, dm, i - clo).XE;
          const double hpw = closed ? t.wh[d - 1] : 0.0;
          if (M <= 4)
            x_cell<4, 4>(lane, xs, M, rowm[kp2].sig, rowm[kp2 + 1].sig, mq.sig, d - 1 >= 4, closed, mh1, maxint, i, j, Tb, MS, gi, em, S,
                         colm.p, cbase, cm.win, hpw, emh, xe, M, xeg);
          else
            x_cell<8, 2>(lane, xs, M, rowm[kp2].sig, rowm[kp2 + 1].sig, mq.sig, d - 1 >= 4, closed, mh1, maxint, i, j, Tb, MS, gi, em, S,
                         colm.p, cbase, cm.win, hpw, emh, xe, M, xeg);
        }
      }
      // ---- cooperative row items: GL consecutive lanes share one row object (a bond row or a left state of one cell), split
      //      its contiguous bond range between them and keep up to 4 column accumulators per pass.
      //      M2 edge ranges | Bl | Br | Z1 | Z2 : weighted dot products of row segments
      {
        const int n9 = nb0;               // M2 edge: bond row of i    x  c  < Sigma_{j+1}
        const int n3 = closed ? nb1 : 0;  // Bl, Br : bond row of p    x  c1 < Sigma_j
        const int n5 = closed ? nl1 : 0;  // Z1     : left state of p  x  c2 < Sigma_q
        const int n6 = closed ? nb2 : 0;  // Z2     : bond row of i+2  x  r  < |R_q|
        const int n2 = 0;                 // (X is advanced by one warp per cell, below)
        const int e9 = n9, e3 = e9 + n3, e4 = e3 + n3, e5 = e4 + n5, e6 = e5 + n6, e2 = e6 + n2;
        const unsigned gmask = GL >= 32 ? 0xffffffffu : ((1u << (GL & 31)) - 1u) << (tid & 31 & ~(GL - 1));
        for (int w; (w = grab(&p1ctr[1])) < (((e2 << LG) + 31) >> 5);) {
          const int ts = (w << 5) + (tid & 31);
          if (ts >= (e2 << LG)) continue;
          const int g = ts >> LG, sub = ts & (GL - 1);
#ifdef CDZ_PHASE_TIMING
          const long long tr0 = clock64();
          const int ttype = g < e9 ? 0 : g < e3 ? 1 : g < e4 ? 2 : g < e5 ? 3 : g < e6 ? 4 : 5;
#endif
          if (g < e6) {
            // ---- decode: out[c] = add[c] + sum_{kb in [lo,hi) (+ [lo2,hi2))} wt[sg * pos(kb) + cst] A[kb] B0[c * S + kb] -------
            const double *A = nullptr, *B0 = nullptr, *wt = nullptr, *addp = nullptr;
            double* out = nullptr;
            const uint8_t* bp = rbp;
            int ncol = 0, lo = 0, hi = 0, lo2 = 0, hi2 = 0, kb0 = rkb0, pb = rbase, sg = 0, cst = 0, nadd = 0;
            double addw = 1.0;
            if (g < e9) {
              const int rr = rb0 + g, kp = rbpos[rr], a = rr - crow[kp];
              const int i = rbase + kp, j = i + d;
              const PosMeta mj1 = colm[j + 1 - cbase];
              const int offi = rowm[kp].off, offj1 = mj1.off;
              ncol = mj1.sig;
              if (I == J) {
                lo = rowm[kp + 1].off;
                hi = offj1;
              } else {
                hi = (I + 1) * CDZ_TB;
                lo = rowm[kp + 1].off < hi ? rowm[kp + 1].off : hi;
                lo2 = J * CDZ_TB;
                hi2 = offj1;
              }
              A = b.QM + (size_t)(offi + a) * S;
              B0 = b.QM1T + (size_t)offj1 * S;
              out = scr_of(scrb, dm, i - clo).M2s + a * M;
              addp = b.GP + (size_t)I * ka.nsplit * (CDZ_TB * CDZ_TB) + (size_t)(offi - I * CDZ_TB + a) * CDZ_TB +
                     (offj1 - J * CDZ_TB);
              nadd = ka.nsplit;
            } else if (g < e4) {
              const bool left = g < e3;
              const int rr = rb1 + (left ? g - e9 : g - e3), kp = rbpos[rr], a1 = rr - crow[kp];
              const int p = rbase + kp, i = p - 1, j = i + d, q = j - 1;
              const PosMeta mj = colm[j - cbase];
              const int offp = rowm[kp].off;
              const int lmax = min(maxint, q - mh1 - p);
              ncol = (pmx[rowm[kp - 1].nuc] & mj.nuc) ? mj.sig : 0;  // nothing to do when no nucleotides of i and j can pair
              wt = cm.wbu;
              if (left) {
                // multiloop closure + left bulges l1 = 2..lmax: E(p,k-1)[a1,s] Qbs(k,q)[s,c1], k = p + l1
                addp = b.M2 + (size_t)(offp + a1) * S + mj.off;
                nadd = 1;
                addw = cm.wac;
                A = b.EM + (size_t)(offp + a1) * S;
                B0 = b.QBST + (size_t)mj.off * S;
                if (lmax >= 2) { lo = rowm[kp + 2].off; hi = rowm[kp + lmax].off + rowm[kp + lmax].sig; }
                sg = 1; cst = -p;
                out = scr_of(scrb, dm, i - clo).Bl + a1 * M;
              } else {
                // right bulges l2 = 2..lmax: Qbs(p,l)[a1,u] E(l+1,q)[u,c1], l = q - l2
                A = b.QBS + (size_t)(offp + a1) * S;
                B0 = b.EMT + (size_t)mj.off * S;
                if (lmax >= 2) { lo = colm[q - lmax + 1 - cbase].off; hi = colm[q - 1 - cbase].off + colm[q - 1 - cbase].sig; }
                bp = cbp; kb0 = ckb0; pb = cbase; sg = -1; cst = j;
                out = scr_of(scrb, dm, i - clo).Br + a1 * M;
              }
            } else if (g < e5) {
              // Z1[lst][c2]: l1 = 1, l2 = 2..lmax: D1(p; l+2)[lst,u] E(l+2,q-1)[u,c2], l = q - l2, weight win[1+l2]
              const int ll = rl1 + (g - e4), kp = rlpos[ll], lst = ll - (rowm[kp].loff - L0);
              const int p = rbase + kp, i = p - 1, j = i + d, q = j - 1;
              const PosMeta mq = colm[q - cbase];
              const int lmax = min(maxint - 1, q - mh1 - (p + 1));
              ncol = (pmx[rowm[kp - 1].nuc] & colm[j - cbase].nuc) ? mq.sig : 0;
              A = b.D1 + (size_t)(rowm[kp].loff + lst) * S;
              B0 = b.EMT + (size_t)mq.off * S;
              if (lmax >= 2) { lo = colm[q - lmax + 2 - cbase].off; hi = mq.off + mq.sig; }
              bp = cbp; kb0 = ckb0; pb = cbase; wt = cm.win; sg = -1; cst = j + 2;
              out = scr_of(scrb, dm, i - clo).Z1 + lst * M;
            } else {
              // Z2[a2][r]: l2 = 1, l1 = 2..lmax: E(p+1,k-2)[a2,s] D2(k-1; q)[s,r], k = p + l1, weight win[l1+1]
              const int rr = rb2 + (g - e5), kp = rbpos[rr], a2 = rr - crow[kp];
              const int i = rbase + kp - 2, p = i + 1, j = i + d, q = j - 1;
              const PosMeta mq = colm[q - cbase];
              const int lmax = min(maxint - 1, (q - 1) - mh1 - p);
              ncol = (pmx[rowm[kp - 2].nuc] & colm[j - cbase].nuc) ? mq.nR : 0;
              A = b.EM + (size_t)(rowm[kp].off + a2) * S;
              B0 = b.D2T + (size_t)mq.roff * S;
              if (lmax >= 2) { lo = rowm[kp].off; hi = rowm[kp + lmax - 2].off + rowm[kp + lmax - 2].sig; }
              wt = cm.win; sg = 1; cst = 2 - p;
              out = scr_of(scrb, dm, i - clo).Z2 + a2 * MR;
            }
            for (int cc = 0; cc < ncol; cc += 4) {
              const int nc4 = min(4, ncol - cc);
              const double* Bc = B0 + (size_t)cc * S;
              // the additive terms of the (up to 4) columns of this pass; lane c of the group takes column c (every lane when GL < 4)
              double add = 0.0, addv[4] = {0.0, 0.0, 0.0, 0.0};
              if (GL >= 4) {
                if (sub < nc4)
                  for (int sp = 0; sp < nadd; ++sp) add += addp[(size_t)sp * (CDZ_TB * CDZ_TB) + cc + sub];
              } else if (sub == 0) {
                for (int sp = 0; sp < nadd; ++sp)
#pragma unroll
                  for (int c = 0; c < 4; ++c)
                    if (c < nc4) addv[c] += addp[(size_t)sp * (CDZ_TB * CDZ_TB) + cc + c];
              }
              double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
              if (wt) {
                const double* B1 = Bc + (nc4 > 1 ? S : 0);
                const double* B2 = Bc + (nc4 > 2 ? 2 * S : 0);
                const double* B3 = Bc + (nc4 > 3 ? 3 * S : 0);
                if (nc4 == 1) {
#pragma unroll 4
                  for (int kb = lo + sub; kb < hi; kb += GL)
                    a0 += wt[sg * (pb + bp[kb - kb0]) + cst] * A[kb] * Bc[kb];
                } else if (nc4 == 2) {
#pragma unroll 4
                  for (int kb = lo + sub; kb < hi; kb += GL) {
                    const double w = wt[sg * (pb + bp[kb - kb0]) + cst] * A[kb];
                    a0 += w * Bc[kb];
                    a1 += w * B1[kb];
                  }
                } else {
#pragma unroll 4
                  for (int kb = lo + sub; kb < hi; kb += GL) {
                    const double w = wt[sg * (pb + bp[kb - kb0]) + cst] * A[kb];
                    a0 += w * Bc[kb];
                    a1 += w * B1[kb];
                    a2 += w * B2[kb];
                    a3 += w * B3[kb];
                  }
                }
              } else {
                const double* B1 = Bc + (nc4 > 1 ? S : 0);
                const double* B2 = Bc + (nc4 > 2 ? 2 * S : 0);
                const double* B3 = Bc + (nc4 > 3 ? 3 * S : 0);
                if (nc4 <= 2) {
#pragma unroll 4
                  for (int kb = lo + sub; kb < hi; kb += GL) { const double w = A[kb]; a0 += w * Bc[kb]; a1 += w * B1[kb]; }
#pragma unroll 4
                  for (int kb = lo2 + sub; kb < hi2; kb += GL) { const double w = A[kb]; a0 += w * Bc[kb]; a1 += w * B1[kb]; }
                } else {
#pragma unroll 4
                  for (int kb = lo + sub; kb < hi; kb += GL) {
                    const double w = A[kb];
                    a0 += w * Bc[kb]; a1 += w * B1[kb]; a2 += w * B2[kb]; a3 += w * B3[kb];
                  }
#pragma unroll 4
                  for (int kb = lo2 + sub; kb < hi2; kb += GL) {
                    const double w = A[kb];
                    a0 += w * Bc[kb]; a1 += w * B1[kb]; a2 += w * B2[kb]; a3 += w * B3[kb];
                  }
                }
              }
#pragma unroll
              for (int o = 1; o < GL; o <<= 1) {
                a0 += __shfl_xor_sync(gmask, a0, o);
                a1 += __shfl_xor_sync(gmask, a1, o);
                a2 += __shfl_xor_sync(gmask, a2, o);
                a3 += __shfl_xor_sync(gmask, a3, o);
              }
              if (GL >= 4) {
                if (sub < nc4) out[cc + sub] = addw * add + (sub == 0 ? a0 : sub == 1 ? a1 : sub == 2 ? a2 : a3);
              } else if (sub == 0) {
                out[cc] = addw * addv[0] + a0;
                if (nc4 > 1) out[cc + 1] = addw * addv[1] + a1;
                if (nc4 > 2) out[cc + 2] = addw * addv[2] + a2;
                if (nc4 > 3) out[cc + 3] = addw * addv[3] + a3;
              }
            }
          }
#ifdef CDZ_PHASE_TIMING
          ttyp[ttype] += clock64() - tr0;
#endif
        }
      }
      CDZ_TICK(0);
      // ---- single-lane items: SB | recursive parts of Qm1, Qml | E(i,j) ----------------------------------------------------
      {
        const int npm = nps << lgM;
        const int n7 = closed ? nb1 * npm : 0;
        const int n8 = nb0 << lgM;
        const int e7 = n7, e8 = e7 + n8, e1 = e8 + n8;
        for (int w; (w = grab(&p1ctr[2])) < ((e1 + 31) >> 5);) {
          const int g = (w << 5) + (tid & 31);
          if (g >= e1) continue;
          if (g < e7) {
            // ---- SB[a'][slot'][c']: inner pair identity kept (stack, bulges of size 1) ------------------------------
            const int rq = g / npm, it = g - rq * npm;
            const int c1 = it & (Mp - 1), sl = it >> lgM, rr = rb1 + rq;
            const int kp = rbpos[rr], a1 = rr - crow[kp];
            const int p = rbase + kp, i = p - 1, j = i + d, q = j - 1;
            const PosMeta mj = colm[j - cbase];
            if (c1 >= mj.sig || !(pmx[rowm[kp - 1].nuc] & mj.nuc)) continue;
            const PosMeta mp = rowm[kp], mq = colm[q - cbase];
            const int xp = cm.slot_x[sl], yp = cm.slot_y[sl];
            // the inner pair (x', y') sits at (p, q), (p+1, q) or (p, q-1): nothing to add when x' or y' cannot occur there
            if (!(((mp.nuc | rowm[kp + 1].nuc) >> xp) & 1) || !(((mq.nuc | colm[q - 1 - cbase].nuc) >> yp) & 1)) {
              scr_of(scrb, dm, i - clo).SB[(a1 * nps + sl) * M + c1] = 0.0;
              continue;
            }
            const int lst = t.lsidx[((size_t)p * MS + a1) * 4 + xp], r = t.rsidx[((size_t)q * 4 + yp) * MS + c1];
            double v = 0.0;
            if (q - p >= mh1 && lst >= 0 && r >= 0) v = b.QB[(size_t)(mp.loff + lst) * RS + mq.roff + r];
            if (maxint >= 1 && q - (p + 1) >= mh1) {
              double s1 = 0.0, s2 = 0.0;
              const PosMeta mp1 = rowm[kp + 1], mq1 = colm[q - 1 - cbase];
              const PosPk wp1 = rowpk[kp + 1], wq1 = colpk[q - 1 - cbase];
              if (FIX) {
                // fixed trip counts + predicates: every global load of the item is in flight before the first product (a skipped term adds 0)
                double tb[4], qa[4], qc[6], tc[6];
#pragma unroll
                for (int l2 = 0; l2 < 4; ++l2) {
                  const bool on = r >= 0 && l2 < mp1.nL && pk(wp1.lsx, l2) == xp;
                  tb[l2] = on ? Tbar[(size_t)p * MS2 + a1 * MS + pk(wp1.lsa, l2)] : 0.0;
                  qa[l2] = on ? b.QB[(size_t)(mp1.loff + l2) * RS + mq.roff + r] : 0.0;
                }
#pragma unroll
                for (int r2 = 0; r2 < 6; ++r2) {
                  const bool on = lst >= 0 && r2 < mq1.nR && pk(wq1.rsy, r2) == yp;
                  qc[r2] = on ? b.QB[(size_t)(mp.loff + lst) * RS + mq1.roff + r2] : 0.0;
                  tc[r2] = on ? Tbar[(size_t)q * MS2 + pk(wq1.rsc, r2) * MS + c1] : 0.0;
                }
#pragma unroll
                for (int l2 = 0; l2 < 4; ++l2) s1 += tb[l2] * qa[l2];
#pragma unroll
                for (int r2 = 0; r2 < 6; ++r2) s2 += qc[r2] * tc[r2];
              } else {
                if (r >= 0) {
                  for (int l2 = 0; l2 < mp1.nL; ++l2)
                    if (pk(wp1.lsx, l2) == xp)
                      s1 += Tbar[(size_t)p * MS2 + a1 * MS + pk(wp1.lsa, l2)] *
                            b.QB[(size_t)(mp1.loff + l2) * RS + mq.roff + r];
                }
                if (lst >= 0) {
                  for (int r2 = 0; r2 < mq1.nR; ++r2)
                    if (pk(wq1.rsy, r2) == yp)
                      s2 += b.QB[(size_t)(mp.loff + lst) * RS + mq1.roff + r2] *
                            Tbar[(size_t)q * MS2 + pk(wq1.rsc, r2) * MS + c1];
                }
              }
              v += cm.wbu[1] * (s1 + s2);
            }
            scr_of(scrb, dm, i - clo).SB[(a1 * nps + sl) * M + c1] = v;
          } else {

            // ---- recursive parts of Qm1 / Qml (g < e8) and E(i,j) (g >= e8) -----------------------------------------
            const bool rec = g < e8;
            const int it = rec ? g - e7 : g - e8;
            const int c = it & (Mp - 1), rr = rb0 + (it >> lgM), kp = rbpos[rr], a = rr - crow[kp];
            const int i = rbase + kp, j = i + d;
            const PosMeta mj1 = colm[j + 1 - cbase];
            if (c >= mj1.sig) continue;
            const PosMeta mj = colm[j - cbase];
            const int offi = rowm[kp].off;
            const double* Tj = Tbar + (size_t)j * MS2 + c;
            if (rec) {
              double r1 = 0.0, r2 = 0.0;
              if (d >= 1) {
                const PosMeta mi1 = rowm[kp + 1];
                const double* Ti = Tbar + (size_t)i * MS2 + a * MS;
                if (FIX) {
                  double q1[4], t1[4], t2[4], q2[4];
#pragma unroll
                  for (int s = 0; s < 4; ++s) {
                    q1[s] = s < mj.sig ? b.QM1T[(size_t)(mj.off + s) * S + offi + a] : 0.0;
                    t1[s] = s < mj.sig ? Tj[s * MS] : 0.0;
                    t2[s] = s < mi1.sig ? Ti[s] : 0.0;
                    q2[s] = s < mi1.sig ? b.QML[(size_t)(mi1.off + s) * S + mj1.off + c] : 0.0;
                  }
#pragma unroll
                  for (int s = 0; s < 4; ++s) { r1 += q1[s] * t1[s]; r2 += t2[s] * q2[s]; }
                } else {
                  for (int s = 0; s < mj.sig; ++s) r1 += b.QM1T[(size_t)(mj.off + s) * S + offi + a] * Tj[s * MS];
                  for (int s = 0; s < mi1.sig; ++s) r2 += Ti[s] * b.QML[(size_t)(mi1.off + s) * S + mj1.off + c];
                }
              }
              Scr sc = scr_of(scrb, dm, i - clo);
              sc.R1[a * M + c] = cm.wb * r1;
              sc.R2[a * M + c] = cm.wb * r2;
            } else {
              double v = 0.0;
              if (FIX) {
                double e1[4], t1[4];
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                  e1[s] = s < mj.sig ? b.EM[(size_t)(offi + a) * S + mj.off + s] : 0.0;
                  t1[s] = s < mj.sig ? Tj[s * MS] : 0.0;
                }
#pragma unroll
                for (int s = 0; s < 4; ++s) v += e1[s] * t1[s];
              } else {
                for (int s = 0; s < mj.sig; ++s) v += b.EM[(size_t)(offi + a) * S + mj.off + s] * Tj[s * MS];
              }
              b.EM[(size_t)(offi + a) * S + mj1.off + c] = v;
              b.EMT[(size_t)(mj1.off + c) * S + offi + a] = v;
            }
          }
        }
      }
      CDZ_TICK(1);
      __syncthreads();
      if (tid == 0) p1ctr[0] = p1ctr[1] = p1ctr[2] = 0;  // every warp has left P1; the next P1 is several barriers away
      CDZ_TICK(2);
      if (closed) {
        // ================= P2: Y[(a',u)][(v,c')] -- everything that carries the closing mismatch =================
        const bool v11 = maxint >= 2 && d - 4 >= mh1;  // 1x1 interior loop: inner pair (p+1, q-1)
        for (int it = tid; it < (nl1 << lgR); it += NT) {
          const int r = it & (MRp - 1), ll = rl1 + (it >> lgR), kp = rlpos[ll], lst = ll - (rowm[kp].loff - L0);
          const int p = rbase + kp, i = p - 1, j = i + d, q = j - 1;
          const PosMeta mq = colm[q - cbase];
          if (r >= mq.nR || !(pmx[rowm[kp - 1].nuc] & colm[j - cbase].nuc)) continue;
          const Scr sc = scr_of(scrb, dm, i - clo);
          const int Sp1 = rowm[kp + 1].sig, Sq = mq.sig;
          const double* TLp = TLs + ((p - tlbase) * ML + lst) * M;
          const double* TRq = TRs + (size_t)(q - trbase) * M * MR + r;
          const double dd11 = v11 ? b.DD[(size_t)(rowm[kp].loff + lst) * RS + mq.roff + r] : 0.0;  // (needed last: the load overlaps the loops)
          double y = 0.0;
          if (FIX) {
            // fixed trip counts + predicates (bond dimension <= 4): all shared-memory operands in flight together; a skipped term adds 0
            double trq[4];
#pragma unroll
            for (int aw = 0; aw < 4; ++aw) trq[aw] = aw < Sq ? TRq[aw * MR] : 0.0;
#pragma unroll
            for (int cz = 0; cz < 4; ++cz) {
              const bool oc = cz < Sp1;
              const double tl = oc ? TLp[cz] : 0.0;
              double s = oc ? sc.Z2[cz * MR + r] : 0.0;
#pragma unroll
              for (int aw = 0; aw < 4; ++aw) s += ((oc && aw < Sq) ? sc.XE[cz * M + aw] : 0.0) * trq[aw];
              y += tl * s;
            }
#pragma unroll
            for (int aw = 0; aw < 4; ++aw) y += (aw < Sq ? sc.Z1[lst * M + aw] : 0.0) * trq[aw];
          } else {
            for (int cz = 0; cz < Sp1; ++cz) {
              const double tl = TLp[cz];
              if (tl == 0.0) continue;
              double s = sc.Z2[cz * MR + r];
              for (int aw = 0; aw < Sq; ++aw) s += sc.XE[cz * M + aw] * TRq[aw * MR];
              y += tl * s;
            }
            for (int aw = 0; aw < Sq; ++aw) y += sc.Z1[lst * M + aw] * TRq[aw * MR];
          }
          sc.Y[lst * MR + r] = cm.win[2] * dd11 + y;
        }
        __syncthreads();
      }
      CDZ_TICK(3);
      // ================= P3b: Qb[(a,x)][(y,c)] = can(x,y) sum T_i[a,x,a'] T_j[c',y,c] inner ============================
      {
        int rl0;
        const int nl0 = ls_rows(clo, chi, rl0);
        for (int it = tid; it < (nl0 << lgR); it += NT) {
          const int r = it & (MRp - 1), ll = rl0 + (it >> lgR), kp = rlpos[ll], lst = ll - (rowm[kp].loff - L0);
          const int i = rbase + kp, j = i + d;
          const PosMeta mj = colm[j - cbase];
          if (r >= mj.nR) continue;
          const Scr sc = scr_of(scrb, dm, i - clo);
          double v = 0.0;
          if (closed) {
            const int x = pk(rowpk[kp].lsx, lst), y = pk(colpk[j - cbase].rsy, r);
            if (cm.pslot[x * 4 + y] >= 0) {
              // Qb = sum_{a',c'} T_i[a,x,a'] T_j[c',y,c] inner[x,y;a',c'] with inner expanded in place (no per-slot table):
              //   inner = Bl + Br + sum_slots wst[P][P'] SB[a'][slot'][c']  +  sum_{(a',u),(v,c')} wtm[P][u][v] Y[(a',u)][(v,c')]
              const int P = cm.ptype[x * 4 + y];
              const PosMeta mp = rowm[kp + 1], mq = colm[j - 1 - cbase];
              const int S1 = mp.sig, S2 = mj.sig;
              const double* TLi = TLs + ((i - tlbase) * ML + lst) * M;
              const double* TRj = TRs + (size_t)(j - trbase) * M * MR + r;
              for (int a1 = 0; a1 < S1; ++a1) {
                const double tl = TLi[a1];
                if (tl == 0.0) continue;
                for (int c1 = 0; c1 < S2; ++c1) {
                  const double tr = TRj[c1 * MR];
                  if (tr == 0.0) continue;
                  double s = sc.Bl[a1 * M + c1] + sc.Br[a1 * M + c1];
                  for (int s2 = 0; s2 < nps; ++s2) s += wsl[P][s2] * sc.SB[(a1 * nps + s2) * M + c1];
                  v += tl * tr * s;
                }
              }
              const PosPk wp = rowpk[kp + 1], wq = colpk[j - 1 - cbase];
              for (int l = 0; l < mp.nL; ++l) {
                const double tl = TLi[pk(wp.lsa, l)];
                if (tl == 0.0) continue;
                const int u = pk(wp.lsx, l);
                double s = 0.0;
                for (int k = 0; k < mq.nR; ++k) s += TRj[pk(wq.rsc, k) * MR] * cm.wtm[P][u][pk(wq.rsy, k)] * sc.Y[l * MR + k];
                v += tl * s;
              }
            }
          }
          sc.QBc[lst * MR + r] = v;
          b.QB[(size_t)(rowm[kp].loff + lst) * RS + mj.roff + r] = v;
        }
      }
      __syncthreads();
      CDZ_TICK(4);
      // ================= P4: Qbs, Qm1, Qml, M2, Qm;  DD = mismatch-dressed extension of Qb(i,j) over [i-1..j+1] ==========
      const bool dress = closed && maxint >= 2;
      int rlm = 0, nlm = 0, rbm = 0, nbm = 0;
      if (dress) {
        // cells with i >= 1 and j <= n-2, i.e. i <= n-2-d
        const int hi = min(chi, n - 2 - d);
        nlm = ls_rows(max(clo, 1) - 1, hi - 1, rlm);
        nbm = bond_rows(max(clo, 1) - 1, hi - 1, rbm);
      }
      {
        const int n4 = nb0 << lgM, n5 = nlm << lgR;
        for (int g = tid; g < n4 + n5; g += NT) {
          if (g < n4) {
            const int c = g & (Mp - 1), rr = rb0 + (g >> lgM), kp = rbpos[rr], a = rr - crow[kp];
            const int i = rbase + kp, j = i + d;
            const PosMeta mj1 = colm[j + 1 - cbase];
            if (c >= mj1.sig) continue;
            const PosMeta mi = rowm[kp], mj = colm[j - cbase];
            const Scr sc = scr_of(scrb, dm, i - clo);
            double qbs = 0.0;
            const unsigned long long wla = rowpk[kp].lsa, wrc = colpk[j - cbase].rsc;
            for (int l = 0; l < mi.nL; ++l)
              if (pk(wla, l) == a)
                for (int k = 0; k < mj.nR; ++k)
                  if (pk(wrc, k) == c) qbs += sc.QBc[l * MR + k];
            const double qm1 = cm.wc * qbs + sc.R1[a * M + c];
            const double qml = qm1 + sc.R2[a * M + c];
            const double m2 = sc.M2s[a * M + c];
            const size_t rc = (size_t)(mi.off + a) * S + mj1.off + c, cr = (size_t)(mj1.off + c) * S + mi.off + a;
            b.QBS[rc] = qbs;
            b.QBST[cr] = qbs;
            b.QM1T[cr] = qm1;
            b.QML[rc] = qml;
            b.M2[rc] = m2;
            b.QM[rc] = qml + m2;
          } else {
            const int it = g - n4;
            const int r = it & (MRp - 1), ll = rlm + (it >> lgR), kp = rlpos[ll], lst = ll - (rowm[kp].loff - L0);
            const int pi = rbase + kp, i = pi + 1, j = i + d, pj = j + 1;
            const PosMeta mpj = colm[pj - cbase];
            if (r >= mpj.nR) continue;
            const PosMeta mi = rowm[kp + 1], mj = colm[j - cbase];
            const Scr sc = scr_of(scrb, dm, i - clo);
            const int up = pk(rowpk[kp].lsx, lst), vp = pk(colpk[pj - cbase].rsy, r);
            const PosPk wi = rowpk[kp + 1], wj = colpk[j - cbase];
            const double* TLm = TLs + ((pi - tlbase) * ML + lst) * M;
            const double* TRp = TRs + (size_t)(pj - trbase) * M * MR + r;
            double v = 0.0;
            for (int l2 = 0; l2 < mi.nL; ++l2) {
              const double tl = TLm[pk(wi.lsa, l2)];
              if (tl == 0.0) continue;
              const int x = pk(wi.lsx, l2);
              double s = 0.0;
              for (int r2 = 0; r2 < mj.nR; ++r2) {
                const int y = pk(wj.rsy, r2);
                if (cm.pslot[x * 4 + y] < 0) continue;
                s += TRp[pk(wj.rsc, r2) * MR] * cm.wtm[cm.ptype[y * 4 + x]][vp][up] * sc.QBc[l2 * MR + r2];
              }
              v += tl * s;
            }
            sc.Y[lst * MR + r] = v;
            b.DD[(size_t)(rowm[kp].loff + lst) * RS + mpj.roff + r] = v;
          }
        }
      }
      __syncthreads();
      CDZ_TICK(5);
      // ================= P5: GI, D1, D2T = DD summed over both / the right / the left nucleotide =========================
      if (dress) {
        // one lane per ROW of the dressed extension (few, longer items): a left state gives its D1 row, a bond row gives its
        // D2T column and its GI row
        for (int g = tid; g < nlm + nbm; g += NT) {
          if (g < nlm) {
            const int ll = rlm + g, kp = rlpos[ll], lst = ll - (rowm[kp].loff - L0);
            const int pi = rbase + kp, i = pi + 1, j = i + d, pj = j + 1;
            const PosMeta mpj = colm[pj - cbase], mpj1 = colm[pj + 1 - cbase];
            const double* y = scr_of(scrb, dm, i - clo).Y + lst * MR;
            double* out = b.D1 + (size_t)(rowm[kp].loff + lst) * S + mpj1.off;
            const unsigned long long wrc = colpk[pj - cbase].rsc;
            for (int c = 0; c < mpj1.sig; ++c) {
              double v = 0.0;
              for (int k = 0; k < mpj.nR; ++k)
                if (pk(wrc, k) == c) v += y[k];
              out[c] = v;
            }
          } else {
            const int rr = rbm + (g - nlm), kp = rbpos[rr], a = rr - crow[kp];
            const int pi = rbase + kp, i = pi + 1, j = i + d, pj = j + 1;
            const PosMeta mpi = rowm[kp], mpj = colm[pj - cbase], mpj1 = colm[pj + 1 - cbase];
            const double* y = scr_of(scrb, dm, i - clo).Y;
            // left states with bond a are contiguous in the (a, x)-sorted list
            int l0 = 0, l1 = 0;
            const unsigned long long wla = rowpk[kp].lsa, wrc = colpk[pj - cbase].rsc;
            for (int l = 0; l < mpi.nL; ++l) {
              const int la = pk(wla, l);
              l0 += la < a;
              l1 += la <= a;
            }
            double gi[CDZ_MAX_BOND];
#pragma unroll
            for (int c = 0; c < CDZ_MAX_BOND; ++c) gi[c] = 0.0;
            for (int k = 0; k < mpj.nR; ++k) {
              double v = 0.0;
              for (int l = l0; l < l1; ++l) v += y[l * MR + k];
              b.D2T[(size_t)(mpj.roff + k) * S + mpi.off + a] = v;
              const int c = pk(wrc, k);
#pragma unroll
              for (int cc = 0; cc < CDZ_MAX_BOND; ++cc) gi[cc] += cc == c ? v : 0.0;
            }
            double* out = b.GI + (size_t)(mpi.off + a) * S + mpj1.off;
#pragma unroll
            for (int c = 0; c < CDZ_MAX_BOND; ++c)
              if (c < mpj1.sig) out[c] = gi[c];
          }
        }
      }
      CDZ_TICK(6);
      // the next phase that writes this scratch (P1 of the next chunk / diagonal) is separated from these reads by the
      // barrier after P1 only for Y; P1 itself writes other arrays, so no barrier is needed here
    }
  }
  // ---- hand the column states (now X_u(i0, j)) to the block above ------------------------------------------------------------
  __syncthreads();
  for (int jc = 0; jc < ncolj; ++jc) {
    const int j = j0 + jc, Sc = xoff[jc + 1] - xoff[jc];
    const double* xs = xst + (size_t)XU * M * xoff[jc];
    double* dst = b.XS + (size_t)j * (XU * MS2);
    for (int e = tid; e < XU * MS * Sc; e += NT) {
      const int c2 = e % Sc, a2 = (e / Sc) % MS, u4 = e / (Sc * MS);
      dst[u4 * MS2 + a2 * MS + c2] = xs[((size_t)u4 * M + a2) * Sc + c2];
    }
  }
#ifdef CDZ_PHASE_TIMING
  if (blockIdx.x == 3 && blockIdx.y == 0 && (tid == 0 || tid == 37 || tid == 300 || tid == 511) && (ka.D == 5 || ka.D == 60 || ka.D == 300))
    printf("D=%d tid=%d coop=%lld single=%lld barwait=%lld P2P3a=%lld P3b=%lld P4=%lld P5=%lld steps=%d | M2=%lld Bl=%lld Br=%lld Z1=%lld Z2=%lld X=%lld\n", ka.D, tid, tph[0], tph[1],
           tph[2], tph[3], tph[4], tph[5], tph[6], dmax - dmin + 1, ttyp[0], ttyp[1], ttyp[2], ttyp[3], ttyp[4], ttyp[5]);
#endif
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int cdz_cell_config(cdz_tables* const* ts, int B, cdz_cell_cfg* cfg) {
  Dims dm{1, 1, 1, 6, 0, 0, 0, 0};
  int maxpos = 1;
  for (int k = 0; k < B; ++k) {
    const cdz_tt* tt = ts[k]->tt;
    dm.M = std::max(dm.M, tt->MS);
    dm.ML = std::max(dm.ML, tt->maxL);
    dm.MR = std::max(dm.MR, tt->maxR);
    dm.nps = std::max(dm.nps, ts[k]->model->c.nps);
    for (int bk = 0; bk < tt->NB; ++bk) maxpos = std::max(maxpos, std::min(tt->blk_start[bk + 1], tt->n + 1) - tt->blk_start[bk]);
  }
  dm.lgM = clog2(dm.M);
  dm.lgR = clog2(dm.MR);
  dm.lgP = clog2(dm.nps);
  int span = 1;
  for (int k = 0; k < B; ++k) {
    const cdz_tt* tt = ts[k]->tt;
    const int n = tt->n;
    for (int bk = 0; bk < tt->NB; ++bk) {
      const int i0 = tt->blk_start[bk], i1 = std::min(tt->blk_start[bk + 1], n);
      const int rbase = std::max(i0 - 1, 0), rend = std::min(i1 + ROWPAD - 2, n);
      span = std::max(span, tt->off[rend] + tt->sigma[rend] - tt->off[rbase]);
      const int j0 = std::max(tt->blk_start[bk], 1) - 1, j1 = tt->blk_start[bk + 1] - 1;
      const int cbase = std::max(j0 - COLPAD + 1, 0), cend = std::min(j1 + 1, n);
      span = std::max(span, tt->off[cend] + tt->sigma[cend] - tt->off[cbase]);
    }
  }
  // dynamic shared memory available to one CTA: the 227 KB opt-in limit minus the static shared memory of the kernel
  cudaFuncAttributes fa0, fa1;
  CDZ_CUDA(cudaFuncGetAttributes(&fa0, cell_kernel<0>));
  CDZ_CUDA(cudaFuncGetAttributes(&fa1, cell_kernel<1>));
  const size_t budget = 227 * 1024 - std::max(fa0.sharedSizeBytes, fa1.sharedSizeBytes) - 256;
  int C = maxpos;
  while (C > 1 && make_plan(maxpos, span, dm, C).total > budget) --C;
  const Plan pl = make_plan(maxpos, span, dm, C);
  if (pl.total > budget) { cdz_set_error("cell kernel: shared-memory need exceeds 200 KB"); return CDZ_ENOMEM; }
  cfg->M = dm.M; cfg->ML = dm.ML; cfg->MR = dm.MR; cfg->nps = dm.nps;
  cfg->maxpos = maxpos; cfg->span = span; cfg->C = C; cfg->smem = pl.total;
  CDZ_CUDA(cudaFuncSetAttribute(cell_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.total));
  CDZ_CUDA(cudaFuncSetAttribute(cell_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.total));
  return CDZ_OK;
}

void cdz_launch_cells(const Ctx* d_ctxs, int B, int nblk, int D, int nsplit, const cdz_cell_cfg* cfg, cudaStream_t st) {
  KArgs ka;
  ka.D = D; ka.nsplit = nsplit; ka.C = cfg->C; ka.maxpos = cfg->maxpos; ka.span = cfg->span;
  ka.dm.M = cfg->M; ka.dm.ML = cfg->ML; ka.dm.MR = cfg->MR; ka.dm.nps = cfg->nps;
  ka.dm.lgM = clog2(cfg->M); ka.dm.lgR = clog2(cfg->MR); ka.dm.lgP = clog2(cfg->nps);
  ka.dm.pc = ka.dm.percell();
  if (cfg->M == 4 && cfg->ML == 4 && cfg->MR == 6 && cfg->nps == 6) cell_kernel<1><<<dim3(nblk, B), CELL_THREADS, cfg->smem, st>>>(d_ctxs, ka);
  else cell_kernel<0><<<dim3(nblk, B), CELL_THREADS, cfg->smem, st>>>(d_ctxs, ka);
}
