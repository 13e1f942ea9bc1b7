// cdz_mfe.cu -- minimisation over sequences and structures (eq 2.8, S4d lines 245-260, Alg S4.5 lines
// 706-749): the inside recursion of DESIGN.md section 3 with every (+, x) of the SumProduct semiring replaced by (min, +) of the tropical
// semiring ("we then swap all operations ... with their equivalents in the tropical semiring (MinSum)", line 260), operator bonuses
// entering as free energies -log x (line 749), followed by an argmin traceback.  The paper has no GPU kernel for this (line 781).
//
//   f(z, s) = E(phi(z), s)/kT - sum_i log x(z_i)   over operator paths z (one operator per position, bonds matching) and structures s;
//   f_min = min f (units of kT, f_min >= -log Z) and one minimiser (sequence, structure).
//
// Layout: the pass reuses the table handle of the inside pass (same workspace carve): QB, QBS(T), QM, QM1T, QML, M2, EM(T), DD, D1, D2T,
// GI, XS, Qext hold the tropical quantities (free energies, CDZ_FINF = none) instead of partition functions; op_x / Tbar hold operator
// costs.  No rescaling is needed (sums of energies grow linearly).  Kernels: mfe_init_kernel; mfe_cell_kernel, one launch per nucleotide
// diagonal d = 0 .. n-1 and one CTA per cell (the pre-contracted form of section 3: dressed extensions, X_u row recursion, all in (min,+));
// mfe_ext_kernel (exterior, serial in j); mfe_trace_kernel (one warp follows the smallest alternative of every decision).
#include <math.h>

#include "cdz_internal.h"

#define CDZ_FINF 1.0e300
#define CDZ_FBIG 1.0e299  // anything above counts as "no state"

namespace {

constexpr int MT = 256;  // threads per CTA
constexpr int MXU = 27;  // interior totals u = 4..30

// loop free energies in units of kT, derived once per CTA from the Boltzmann factors of the model (g = -log w)
struct GModel {
  double gst[6][6], gtm[6][4][4], gbu[32], gin[32], ga_c, gb, gc;
};

__device__ __forceinline__ double fmin2(double a, double b) { return a < b ? a : b; }

__device__ __forceinline__ void smem_min(double* addr, double v) {  // atomic min on a shared / global double
  unsigned long long* p = (unsigned long long*)addr;
  unsigned long long old = *p;
  while (v < __longlong_as_double((long long)old)) {
    const unsigned long long assumed = old;
    old = atomicCAS(p, assumed, (unsigned long long)__double_as_longlong(v));
    if (old == assumed) break;
  }
}

__device__ void load_gmodel(GModel* g, const CModel* cm) {
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int k = tid; k < 36; k += nt) g->gst[k / 6][k % 6] = -log(cm->wst[k / 6][k % 6]);
  for (int k = tid; k < 96; k += nt) (&g->gtm[0][0][0])[k] = -log((&cm->wtm[0][0][0])[k]);
  for (int k = tid; k < 32; k += nt) {
    g->gbu[k] = (k >= 1 && k <= 30) ? -log(cm->wbu[k]) : CDZ_FINF;
    g->gin[k] = (k >= 2 && k <= 30) ? -log(cm->win[k]) : CDZ_FINF;
  }
  if (tid == 0) { g->ga_c = -log(cm->wac); g->gb = -log(cm->wb); g->gc = -log(cm->wc); }
}

// every table entry = "none"; operator costs; transfer costs Tbar[i][a][c] = min over the operators (a, ., c); E(i,i-1) = identity (0)
__global__ void mfe_init_kernel(const Ctx* ctx) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const int n = t.n, MS = t.MS, MS2 = MS * MS;
  const size_t S = (size_t)t.S, LS = (size_t)t.LS, RS = (size_t)t.RS;
  const size_t stride = (size_t)gridDim.x * blockDim.x, k0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  double* ss[] = {b.GI, b.QBS, b.QM, b.QM1T, b.QML, b.M2, b.EM, b.EMT, b.QBST};
  for (int w = 0; w < 9; ++w)
    for (size_t k = k0; k < S * S; k += stride) ss[w][k] = CDZ_FINF;
  for (size_t k = k0; k < LS * RS; k += stride) { b.QB[k] = CDZ_FINF; b.DD[k] = CDZ_FINF; }
  for (size_t k = k0; k < LS * S; k += stride) b.D1[k] = CDZ_FINF;
  for (size_t k = k0; k < RS * S; k += stride) b.D2T[k] = CDZ_FINF;
  for (size_t k = k0; k < (size_t)n * MXU * MS2; k += stride) b.XS[k] = CDZ_FINF;
  for (size_t k = k0; k < S; k += stride) b.Qext[k] = CDZ_FINF;
  for (size_t k = k0; k < (size_t)t.opstart[n]; k += stride) t.op_x[k] = -log(t.op_x0[k]);
  for (size_t k = k0; k < (size_t)n * MS2; k += stride) t.Tbar[k] = CDZ_FINF;
}
__global__ void mfe_init2_kernel(const Ctx* ctx) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const int n = t.n, MS = t.MS;
  const size_t S = (size_t)t.S;
  const size_t stride = (size_t)gridDim.x * blockDim.x, k0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t k = k0; k < S; k += stride) { b.EM[k * S + k] = 0.0; b.EMT[k * S + k] = 0.0; }
  for (size_t i = k0; i < (size_t)n; i += stride)
    for (int z = t.opstart[i]; z < t.opstart[i + 1]; ++z) {
      double* e = &t.Tbar[(i * MS + t.op_a[z]) * MS + t.op_c[z]];
      *e = fmin2(*e, t.op_x[z]);
    }
  if (k0 == 0) b.Qext[0] = 0.0;  // Fext(-1) = [0]
}

// shared-memory plan of mfe_cell_kernel (doubles)
struct MPlan { int tl, tr, xo, xn, xe, bl, br, z1, z2, sb, y, inn, qb, res, total; };
__host__ __device__ inline MPlan mplan(int MS, int ML, int MR, int nps) {
  MPlan p;
  const int MS2 = MS * MS;
  int o = 0;
  auto take = [&](int k) { int r = o; o += (k + 1) & ~1; return r; };
  p.tl = take(3 * ML * MS); p.tr = take(3 * MS * MR);
  p.xo = take(MXU * MS2); p.xn = take(MXU * MS2); p.xe = take(MS2);
  p.bl = take(MS2); p.br = take(MS2); p.z1 = take(ML * MS); p.z2 = take(MS * MR);
  p.sb = take(nps * MS2); p.y = take(ML * MR); p.inn = take(nps * MS2); p.qb = take(ML * MR);
  p.res = take(5 * MS2);
  p.total = o;
  return p;
}

// one cell (i, j = i + d) of the tropical pass
__global__ void __launch_bounds__(MT) mfe_cell_kernel(const Ctx* ctx, int d, int ML, int MR) {
  extern __shared__ double msm[];
  __shared__ GModel g;
  __shared__ int offW[2][72], sigW[2][72];
  __shared__ uint8_t sLa[3][CDZ_MAX_STATES], sLx[3][CDZ_MAX_STATES], sRy[3][CDZ_MAX_STATES], sRc[3][CDZ_MAX_STATES];
  __shared__ int snL[3], snR[3];
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const CModel& m = *ctx->cm;
  const int n = t.n, MS = t.MS, MS2 = MS * MS, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const size_t S = (size_t)t.S, RS = (size_t)t.RS;
  const int nps = m.nps;
  const MPlan pl = mplan(MS, ML, MR, nps);
  double *TL = msm + pl.tl, *TR = msm + pl.tr, *xo = msm + pl.xo, *xn = msm + pl.xn, *xe = msm + pl.xe, *bl = msm + pl.bl,
         *br = msm + pl.br, *z1 = msm + pl.z1, *z2 = msm + pl.z2, *sb = msm + pl.sb, *y = msm + pl.y, *inn = msm + pl.inn,
         *qb = msm + pl.qb, *res = msm + pl.res;
  double *TLm = TL, *TLi = TL + ML * MS, *TLp = TLi + ML * MS;   // cost cores T_{i-1}, T_i, T_{i+1}: [lst][c]
  double *TRq = TR, *TRj = TR + MS * MR, *TRn = TRj + MS * MR;   // T_{j-1}, T_j, T_{j+1}: [a][r]
  const int i = blockIdx.x, j = i + d, p = i + 1, q = j - 1;
  const int mh1 = m.min_hairpin + 1, MI = m.max_interior;
  const bool closed = d >= mh1;
  load_gmodel(&g, &m);
  if (tid < 144) {
    const int which = tid / 72, idx = tid % 72, pos = (which ? j : i) - 35 + idx;
    const bool ok = pos >= 0 && pos <= n;
    offW[which][idx] = ok ? t.off[pos] : 0;
    sigW[which][idx] = ok ? t.sig[pos] : 0;
  }
  if (tid >= 160 && tid < 160 + 6 * CDZ_MAX_STATES) {
    const int w6 = (tid - 160) / CDZ_MAX_STATES, k = (tid - 160) % CDZ_MAX_STATES;
    const int pos = w6 < 3 ? i - 1 + w6 : j - 1 + (w6 - 3);
    const bool ok = pos >= 0 && pos < n;
    if (w6 < 3) {
      const int l0 = ok ? t.loff[pos] : 0, nl = ok ? t.loff[pos + 1] - l0 : 0;
      if (k < nl) { sLa[w6][k] = t.ls_a[l0 + k]; sLx[w6][k] = t.ls_x[l0 + k]; }
      if (k == 0) snL[w6] = nl;
    } else {
      const int r0 = ok ? t.roff[pos] : 0, nr = ok ? t.roff[pos + 1] - r0 : 0;
      if (k < nr) { sRy[w6 - 3][k] = t.rs_y[r0 + k]; sRc[w6 - 3][k] = t.rs_c[r0 + k]; }
      if (k == 0) snR[w6 - 3] = nr;
    }
  }
  for (int k = tid; k < 3 * ML * MS + 3 * MS * MR; k += MT) (k < 3 * ML * MS ? TL[k] : TR[k - 3 * ML * MS]) = CDZ_FINF;
  __syncthreads();
  auto offA = [&](int pos) { return offW[0][pos - i + 35]; };
  auto sigA = [&](int pos) { return sigW[0][pos - i + 35]; };
  auto offB = [&](int pos) { return offW[1][pos - j + 35]; };
  auto sigB = [&](int pos) { return sigW[1][pos - j + 35]; };
  // min-plus stretch E(pp,qq)[a][c] with pp and qq+1 near j
  auto FBn = [&](int pp, int qq, int a, int c) { return qq < pp ? (a == c ? 0.0 : CDZ_FINF) : b.EM[(size_t)(offB(pp) + a) * S + offB(qq + 1) + c]; };
  for (int e = tid; e < 6 * 64; e += MT) {
    const int w6 = e / 64, k = e % 64;
    const int pos = w6 < 3 ? i - 1 + w6 : j - 1 + (w6 - 3);
    if (pos < 0 || pos >= n) continue;
    const int z0 = t.opstart[pos], nz = t.opstart[pos + 1] - z0;
    for (int zz = k; zz < nz; zz += 64) {
      const int z = z0 + zz;
      if (w6 < 3) smem_min(&TL[w6 * ML * MS + t.op_l[z] * MS + t.op_c[z]], t.op_x[z]);
      else smem_min(&TR[(w6 - 3) * MS * MR + t.op_a[z] * MR + t.op_r[z]], t.op_x[z]);
    }
  }
  const int Si = sigA(i), Sj1 = sigB(j + 1), offi = offA(i), offj1 = offB(j + 1), nent = Si * Sj1;
  const int offj = offB(j), Sj = sigB(j);
  // ---- E(i,j) = E(i,j-1) (x) Tbar_j ---------------------------------------------------------------------------------------------------
  if (tid < nent) {
    const int a = tid / Sj1, c = tid % Sj1;
    double v = CDZ_FINF;
    for (int s = 0; s < Sj; ++s) v = fmin2(v, b.EM[(size_t)(offi + a) * S + offj + s] + t.Tbar[((size_t)j * MS + s) * MS + c]);
    b.EM[(size_t)(offi + a) * S + offj1 + c] = v;
    b.EMT[(size_t)(offj1 + c) * S + offi + a] = v;
  }
  __syncthreads();
  // ---- interior-loop bodies X_u(i,j), u = 4..30, in place in the state of column j; XE = min_u g_In(u) + X_u, and the hairpin ---------
  const int Sp1 = d >= 2 ? sigA(i + 2) : 0, Sq = d >= 2 ? sigB(j - 1) : 0;
  if (d >= 4) {
    double* xs = b.XS + (size_t)j * (MXU * MS2);
    for (int e = tid; e < MXU * MS2; e += MT) xo[e] = xs[e];
    __syncthreads();
    const int S3 = sigA(i + 3);
    for (int e = tid; e < MXU * MS2; e += MT) {
      const int u4 = e / MS2, a = (e % MS2) / MS, c = e % MS, u = u4 + 4;
      double v = CDZ_FINF;
      if (a < Sp1 && c < Sq) {
        if (u4 > 0 && d - 1 >= 4)
          for (int a3 = 0; a3 < S3; ++a3) v = fmin2(v, t.Tbar[((size_t)(i + 2) * MS + a) * MS + a3] + xo[(u4 - 1) * MS2 + a3 * MS + c]);
        if (d - 2 - u >= mh1) {
          const int l = j + 1 - u, Su = sigB(l + 2);
          const double* gi = b.GI + (size_t)(offA(i + 2) + a) * S + offB(l + 2);
          for (int u2 = 0; u2 < Su; ++u2) v = fmin2(v, gi[u2] + FBn(l + 2, j - 2, u2, c));
        }
      }
      xn[e] = v;
      xs[e] = v;
    }
    __syncthreads();
  }
  if (closed)
    for (int e = tid; e < MS2; e += MT) {
      const int a = e / MS, c = e % MS;
      double v = CDZ_FINF;
      if (a < Sp1 && c < Sq) {
        v = -log(t.wh[d - 1]) + b.EM[(size_t)(offA(i + 2) + a) * S + offB(j - 1) + c];  // hairpin: g_H(d-1) + E(i+2, j-2)
        if (d >= 4)
          for (int u4 = 0; u4 < MXU; ++u4)
            if (u4 + 4 <= MI) v = fmin2(v, g.gin[u4 + 4] + xn[u4 * MS2 + e]);
      }
      xe[e] = v;
    }
  __syncthreads();
  const int nL = snL[1], nR = snR[1], npair = nL * nR, Li0 = t.loff[i], Rj0 = t.roff[j];
  const int Sa = d >= 1 ? sigA(p) : 0, Sc = Sj;  // a' in Sigma_{i+1}, c' in Sigma_j
  const int nLp = snL[2], nRq = snR[0], Lp0 = d >= 1 ? t.loff[p] : 0, Rq0 = d >= 1 ? t.roff[q] : 0;
  const int offp = offA(p), offp1 = offA(p + 1), offq = d >= 1 ? offB(q) : 0;
  if (closed) {
    // ---- Bl, Br, Z1, Z2 (band minima), SB -----------------------------------------------------------------------------------------------
    const int lmaxB = min(MI, q - mh1 - p), lmaxZ1 = min(MI - 1, q - mh1 - (p + 1)), lmaxZ2 = min(MI - 1, (q - 1) - mh1 - p);
    const int nb = Sa * Sc, nz1 = nLp * Sq, nz2 = Sp1 * nRq;
    for (int e = tid; e < 2 * nb + nz1 + nz2; e += MT) {
      const double *A_, *B_, *wt;
      int lo, hi, near_i, base_pos, sgn;
      double v = CDZ_FINF;
      double* out;
      if (e < nb) {
        const int a1 = e / Sc, c1 = e % Sc;
        v = g.ga_c + b.M2[(size_t)(offp + a1) * S + offj + c1];
        A_ = b.EM + (size_t)(offp + a1) * S; B_ = b.QBST + (size_t)(offj + c1) * S;
        lo = p + 2; hi = p + lmaxB; near_i = 1; wt = g.gbu; base_pos = p; sgn = 1;
        out = bl + a1 * MS + c1;
      } else if (e < 2 * nb) {
        const int a1 = (e - nb) / Sc, c1 = (e - nb) % Sc;
        A_ = b.QBS + (size_t)(offp + a1) * S; B_ = b.EMT + (size_t)(offj + c1) * S;
        lo = q - lmaxB + 1; hi = q - 1; near_i = 0; wt = g.gbu; base_pos = j; sgn = -1;
        out = br + a1 * MS + c1;
      } else if (e < 2 * nb + nz1) {
        const int f = e - 2 * nb, lst = f / Sq, c2 = f % Sq;
        A_ = b.D1 + (size_t)(Lp0 + lst) * S; B_ = b.EMT + (size_t)(offq + c2) * S;
        lo = q - lmaxZ1 + 2; hi = q; near_i = 0; wt = g.gin; base_pos = j + 2; sgn = -1;
        out = z1 + lst * MS + c2;
      } else {
        const int f = e - 2 * nb - nz1, a2 = f / nRq, r = f % nRq;
        A_ = b.EM + (size_t)(offp1 + a2) * S; B_ = b.D2T + (size_t)(Rq0 + r) * S;
        lo = p + 1; hi = p + lmaxZ2 - 1; near_i = 1; wt = g.gin; base_pos = p - 2; sgn = 1;
        out = z2 + a2 * MR + r;
      }
      for (int pos = lo; pos <= hi; ++pos) {
        const int o = near_i ? offA(pos) : offB(pos), sg = near_i ? sigA(pos) : sigB(pos);
        double s_ = CDZ_FINF;
        for (int kb = o; kb < o + sg; ++kb) s_ = fmin2(s_, A_[kb] + B_[kb]);
        v = fmin2(v, wt[sgn * (pos - base_pos)] + s_);
      }
      *out = v;
    }
    for (int e = tid; e < nps * Sa * Sc; e += MT) {
      const int sl = e / (Sa * Sc), a1 = (e % (Sa * Sc)) / Sc, c1 = e % Sc;
      const int xp = m.slot_x[sl], yp = m.slot_y[sl];
      const int lst = t.lsidx[((size_t)p * MS + a1) * 4 + xp], r = t.rsidx[((size_t)q * 4 + yp) * MS + c1];
      double v = CDZ_FINF;
      if (q - p >= mh1 && lst >= 0 && r >= 0) v = b.QB[(size_t)(Lp0 + lst) * RS + Rq0 + r];
      if (MI >= 1 && q - (p + 1) >= mh1) {
        double s1 = CDZ_FINF, s2 = CDZ_FINF;
        if (r >= 0)
          for (int l2 = t.loff[p + 1]; l2 < t.loff[p + 2]; ++l2)
            if (t.ls_x[l2] == xp) s1 = fmin2(s1, t.Tbar[((size_t)p * MS + a1) * MS + t.ls_a[l2]] + b.QB[(size_t)l2 * RS + Rq0 + r]);
        if (lst >= 0)
          for (int r2 = t.roff[q - 1]; r2 < t.roff[q]; ++r2)
            if (t.rs_y[r2] == yp) s2 = fmin2(s2, b.QB[(size_t)(Lp0 + lst) * RS + r2] + t.Tbar[((size_t)q * MS + t.rs_c[r2]) * MS + c1]);
        v = fmin2(v, g.gbu[1] + fmin2(s1, s2));
      }
      sb[sl * MS2 + a1 * MS + c1] = v;
    }
    __syncthreads();
    // ---- Y[lst][r]: everything that carries the closing mismatch -------------------------------------------------------------------
    {
      const bool v11 = MI >= 2 && d - 4 >= mh1;
      for (int e = tid; e < nLp * nRq; e += MT) {
        const int lst = e / nRq, r = e % nRq;
        double v = v11 ? g.gin[2] + b.DD[(size_t)(Lp0 + lst) * RS + Rq0 + r] : CDZ_FINF;
        for (int cz = 0; cz < Sp1; ++cz) {
          const double tl = TLp[lst * MS + cz];
          if (tl >= CDZ_FBIG) continue;
          double s_ = z2[cz * MR + r];
          for (int aw = 0; aw < Sq; ++aw) s_ = fmin2(s_, xe[cz * MS + aw] + TRq[aw * MR + r]);
          v = fmin2(v, tl + s_);
        }
        for (int aw = 0; aw < Sq; ++aw) v = fmin2(v, z1[lst * MS + aw] + TRq[aw * MR + r]);
        y[lst * MR + r] = v;
      }
    }
    __syncthreads();
    // ---- inner[slot][a1][c1] ---------------------------------------------------------------------------------------------------------------
    for (int e = tid; e < nps * Sa * Sc; e += MT) {
      const int sl = e / (Sa * Sc), a1 = (e % (Sa * Sc)) / Sc, c1 = e % Sc;
      const int P = m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]];
      double v = fmin2(bl[a1 * MS + c1], br[a1 * MS + c1]);
      for (int s2 = 0; s2 < nps; ++s2) v = fmin2(v, g.gst[P][m.ptype[m.slot_x[s2] * 4 + m.slot_y[s2]]] + sb[s2 * MS2 + a1 * MS + c1]);
      for (int lst = 0; lst < nLp; ++lst) {
        if (sLa[2][lst] != a1) continue;
        const int u = sLx[2][lst];
        for (int r = 0; r < nRq; ++r)
          if (sRc[0][r] == c1) v = fmin2(v, g.gtm[P][u][sRy[0][r]] + y[lst * MR + r]);
      }
      inn[sl * MS2 + a1 * MS + c1] = v;
    }
    __syncthreads();
  }
  // ---- Qb[(a,x)][(y,c)] = T_i (x) T_j (x) inner ----------------------------------------------------------------------------------------
  for (int e = tid; e < npair; e += MT) {
    const int l = e / nR, r = e % nR;
    double v = CDZ_FINF;
    if (closed) {
      const int sl = m.pslot[sLx[1][l] * 4 + sRy[1][r]];
      if (sl >= 0)
        for (int a1 = 0; a1 < Sa; ++a1) {
          const double tl = TLi[l * MS + a1];
          if (tl >= CDZ_FBIG) continue;
          for (int c1 = 0; c1 < Sc; ++c1) v = fmin2(v, tl + TRj[c1 * MR + r] + inn[sl * MS2 + a1 * MS + c1]);
        }
    }
    if (v >= CDZ_FBIG) v = CDZ_FINF;
    qb[l * MR + r] = v;
    b.QB[(size_t)(Li0 + l) * RS + Rj0 + r] = v;
  }
  __syncthreads();
  // ---- Qbs, Qm1, Qml, M2 (split-point minimum over the bonds between i and j), Qm ---------------------------------------------------------
  double* fm2 = res + 4 * MS2;
  for (int e = warp; e < nent; e += MT / 32) {
    const int a = e / Sj1, c = e % Sj1;
    const double* A_ = b.QM + (size_t)(offi + a) * S;
    const double* B_ = b.QM1T + (size_t)(offj1 + c) * S;
    double v = CDZ_FINF;
    for (int kb = (d >= 1 ? offA(i + 1) : offj1) + lane; kb < offj1; kb += 32) v = fmin2(v, A_[kb] + B_[kb]);
    for (int o = 16; o > 0; o >>= 1) v = fmin2(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) fm2[e] = v >= CDZ_FBIG ? CDZ_FINF : v;
  }
  __syncthreads();
  if (tid < nent) {
    const int a = tid / Sj1, c = tid % Sj1;
    double fbs = CDZ_FINF;
    for (int l = 0; l < nL; ++l)
      if (sLa[1][l] == a)
        for (int r = 0; r < nR; ++r)
          if (sRc[1][r] == c) fbs = fmin2(fbs, qb[l * MR + r]);
    double fm1 = g.gc + fbs, fml;
    if (d >= 1)
      for (int s_ = 0; s_ < Sj; ++s_) fm1 = fmin2(fm1, g.gb + b.QM1T[(size_t)(offj + s_) * S + offi + a] + t.Tbar[((size_t)j * MS + s_) * MS + c]);
    fml = fm1;
    if (d >= 1)
      for (int s_ = 0; s_ < Sa; ++s_) fml = fmin2(fml, g.gb + t.Tbar[((size_t)i * MS + a) * MS + s_] + b.QML[(size_t)(offp + s_) * S + offj1 + c]);
    if (fm1 >= CDZ_FBIG) fm1 = CDZ_FINF;
    if (fml >= CDZ_FBIG) fml = CDZ_FINF;
    const size_t rc = (size_t)(offi + a) * S + offj1 + c, cr = (size_t)(offj1 + c) * S + offi + a;
    b.QBS[rc] = fbs;
    b.QBST[cr] = fbs;
    b.QM1T[cr] = fm1;
    b.QML[rc] = fml;
    b.M2[rc] = fm2[tid];
    b.QM[rc] = fmin2(fml, fm2[tid]);
  }
  // ---- dressed extension of Qb(i,j) over [i-1 .. j+1]: DD, and its minima over one / both nucleotides D1, D2T, GI -----------------------
  if (closed && MI >= 2 && i >= 1 && j <= n - 2) {
    const int nLm = snL[0], nRn = snR[2], Lm0 = t.loff[i - 1], Rn0 = t.roff[j + 1];
    double* dd = y;  // (Y is no longer needed)
    __syncthreads();
    for (int e = tid; e < nLm * nRn; e += MT) {
      const int lst = e / nRn, r = e % nRn;
      const int up = sLx[0][lst], vp = sRy[2][r];
      double v = CDZ_FINF;
      for (int l2 = 0; l2 < nL; ++l2) {
        const double tl = TLm[lst * MS + sLa[1][l2]];
        if (tl >= CDZ_FBIG) continue;
        const int x = sLx[1][l2];
        for (int r2 = 0; r2 < nR; ++r2) {
          const int yy = sRy[1][r2];
          if (m.pslot[x * 4 + yy] < 0) continue;
          v = fmin2(v, tl + TRn[sRc[1][r2] * MR + r] + g.gtm[m.ptype[yy * 4 + x]][vp][up] + qb[l2 * MR + r2]);
        }
      }
      if (v >= CDZ_FBIG) v = CDZ_FINF;
      dd[lst * MR + r] = v;
      b.DD[(size_t)(Lm0 + lst) * RS + Rn0 + r] = v;
    }
    __syncthreads();
    const int Sm = sigA(i - 1), Sn2 = sigB(j + 2), offm = offA(i - 1), offn2 = offB(j + 2);
    for (int e = tid; e < nLm * Sn2 + nRn * Sm + Sm * Sn2; e += MT) {
      double v = CDZ_FINF;
      if (e < nLm * Sn2) {
        const int lst = e / Sn2, c = e % Sn2;
        for (int r = 0; r < nRn; ++r)
          if (sRc[2][r] == c) v = fmin2(v, dd[lst * MR + r]);
        b.D1[(size_t)(Lm0 + lst) * S + offn2 + c] = v;
      } else if (e < nLm * Sn2 + nRn * Sm) {
        const int f = e - nLm * Sn2, r = f / Sm, a = f % Sm;
        for (int lst = 0; lst < nLm; ++lst)
          if (sLa[0][lst] == a) v = fmin2(v, dd[lst * MR + r]);
        b.D2T[(size_t)(Rn0 + r) * S + offm + a] = v;
      } else {
        const int f = e - nLm * Sn2 - nRn * Sm, a = f / Sn2, c = f % Sn2;
        for (int lst = 0; lst < nLm; ++lst)
          if (sLa[0][lst] == a)
            for (int r = 0; r < nRn; ++r)
              if (sRc[2][r] == c) v = fmin2(v, dd[lst * MR + r]);
        b.GI[(size_t)(offm + a) * S + offn2 + c] = v;
      }
    }
  }
}

// exterior: Fext(j)[c] = min( Fext(j-1) (x) Tbar_j,  min_{kb < off[j+1]} Fext_bond[kb] + Qbs[kb][(j+1,c)] ), serial in j (one CTA)
__global__ void __launch_bounds__(1024) mfe_ext_kernel(const Ctx* ctx) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const int n = t.n, MS = t.MS;
  const size_t S = (size_t)t.S;
  __shared__ double part[32][CDZ_MAX_BOND];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  for (int j = 0; j < n; ++j) {
    const int Sj1 = t.sig[j + 1], Sj = t.sig[j], oj1 = t.off[j + 1], oj = t.off[j];
    const int len = oj1, per = (len + nwarp - 1) / nwarp, w0 = warp * per, w1 = min(len, w0 + per);
    for (int c = 0; c < Sj1; ++c) {
      const double* q = b.QBST + (size_t)(oj1 + c) * S;
      double v = CDZ_FINF;
      for (int kb = w0 + lane; kb < w1; kb += 32) v = fmin2(v, b.Qext[kb] + q[kb]);
      for (int o = 16; o > 0; o >>= 1) v = fmin2(v, __shfl_xor_sync(0xffffffffu, v, o));
      if (lane == 0) part[warp][c] = v;
    }
    __syncthreads();
    if (tid < Sj1) {
      double v = CDZ_FINF;
      for (int w = 0; w < nwarp; ++w) v = fmin2(v, part[w][tid]);
      for (int s_ = 0; s_ < Sj; ++s_) v = fmin2(v, b.Qext[oj + s_] + t.Tbar[((size_t)j * MS + s_) * MS + tid]);
      b.Qext[oj1 + tid] = v >= CDZ_FBIG ? CDZ_FINF : v;
    }
    __syncthreads();
  }
  if (tid == 0) {
    double best = CDZ_FINF;
    for (int c = 0; c < t.sig[n]; ++c) best = fmin2(best, b.Qext[t.off[n] + c]);
    b.result[0] = best;
  }
}

// ------------------------------------------------------------------------------------------------------------------------------------------------
// argmin traceback (one warp): every decision evaluates its alternatives from the stored tropical tables and follows the smallest
// ------------------------------------------------------------------------------------------------------------------------------------------------
struct MItem { int type, i, j; short a, x, y, c; };
enum { MI_QB = 0, MI_QM = 1, MI_QML = 2, MI_QM1 = 3 };

template <typename F>
__device__ __forceinline__ int warp_argmin(int lane, int count, F value, double* vout = nullptr) {
  double bv = CDZ_FINF;
  int bi = 0x7fffffff;
  for (int idx = lane; idx < count; idx += 32) {
    const double v = value(idx);
    if (v < bv) { bv = v; bi = idx; }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
  if (vout) *vout = bv;
  return bi;
}

struct MV {
  const DevTT& t;
  const DevTab& b;
  const CModel& m;
  const GModel& g;
  __device__ double E(int p, int q, int a, int c) const {
    if (q < p) return a == c ? 0.0 : CDZ_FINF;
    return b.EM[(size_t)(t.off[p] + a) * t.S + t.off[q + 1] + c];
  }
  __device__ double QB(int i, int j, int a, int x, int y, int c) const {
    const int ll = t.lsidx[((size_t)i * t.MS + a) * 4 + x], rr = t.rsidx[((size_t)j * 4 + y) * t.MS + c];
    if (ll < 0 || rr < 0) return CDZ_FINF;
    return b.QB[(size_t)(t.loff[i] + ll) * t.RS + t.roff[j] + rr];
  }
  __device__ bool can(int x, int y) const { return m.pslot[x * 4 + y] >= 0; }
  __device__ int pt(int x, int y) const { return m.ptype[x * 4 + y]; }
};

// smallest value of the loop closed by (i,j) [pair type P, inner bonds ap / cp] with inner pair (k,l), from the dressed tables
__device__ double mfe_loop_value(const MV& V, int i, int j, int k, int l, int P, int ap, int cp) {
  const DevTT& t = V.t;
  const DevTab& b = V.b;
  const CModel& m = V.m;
  const GModel& g = V.g;
  const int l1 = k - i - 1, l2 = j - l - 1, MS = t.MS;
  const size_t S = (size_t)t.S, RS = (size_t)t.RS;
  double best = CDZ_FINF;
  if (l1 == 0 && l2 == 0) {
    for (int sl = 0; sl < m.nps; ++sl) best = fmin2(best, g.gst[P][V.pt(m.slot_x[sl], m.slot_y[sl])] + V.QB(k, l, ap, m.slot_x[sl], m.slot_y[sl], cp));
    return best;
  }
  if (l1 == 0 || l2 == 0) {
    const int len = l1 + l2;
    if (len >= 2) {
      if (l2 == 0) { for (int s = 0; s < t.sig[k]; ++s) best = fmin2(best, V.E(i + 1, k - 1, ap, s) + b.QBS[(size_t)(t.off[k] + s) * S + t.off[l + 1] + cp]); }
      else { for (int u = 0; u < t.sig[l + 1]; ++u) best = fmin2(best, b.QBS[(size_t)(t.off[k] + ap) * S + t.off[l + 1] + u] + V.E(l + 1, j - 1, u, cp)); }
      return g.gbu[len] + best;
    }
    for (int sl = 0; sl < m.nps; ++sl) {
      const int xp = m.slot_x[sl], yp = m.slot_y[sl];
      double q = CDZ_FINF;
      if (l2 == 0) { for (int s = 0; s < t.sig[k]; ++s) q = fmin2(q, t.Tbar[((size_t)(i + 1) * MS + ap) * MS + s] + V.QB(k, l, s, xp, yp, cp)); }
      else { for (int u = 0; u < t.sig[l + 1]; ++u) q = fmin2(q, V.QB(k, l, ap, xp, yp, u) + t.Tbar[((size_t)(j - 1) * MS + u) * MS + cp]); }
      best = fmin2(best, g.gst[P][V.pt(xp, yp)] + q);
    }
    return g.gbu[1] + best;
  }
  const int pl = k - 1, pr = l + 1;
  if (l1 == 1 && l2 == 1) {
    for (int lst = t.loff[pl]; lst < t.loff[pl + 1]; ++lst) {
      if (t.ls_a[lst] != ap) continue;
      for (int r = t.roff[pr]; r < t.roff[pr + 1]; ++r)
        if (t.rs_c[r] == cp) best = fmin2(best, g.gtm[P][t.ls_x[lst]][t.rs_y[r]] + b.DD[(size_t)lst * RS + r]);
    }
  } else if (l1 == 1) {
    for (int lst = t.loff[pl]; lst < t.loff[pl + 1]; ++lst) {
      if (t.ls_a[lst] != ap) continue;
      const double* d1 = b.D1 + (size_t)lst * S + t.off[l + 2];
      for (int w = t.opstart[j - 1]; w < t.opstart[j]; ++w) {
        if (t.op_c[w] != cp) continue;
        double s = CDZ_FINF;
        for (int t2 = 0; t2 < t.sig[l + 2]; ++t2) s = fmin2(s, d1[t2] + V.E(l + 2, j - 2, t2, t.op_a[w]));
        best = fmin2(best, t.op_x[w] + g.gtm[P][t.ls_x[lst]][t.op_b[w]] + s);
      }
    }
  } else if (l2 == 1) {
    for (int r = t.roff[pr]; r < t.roff[pr + 1]; ++r) {
      if (t.rs_c[r] != cp) continue;
      const double* d2 = b.D2T + (size_t)r * S + t.off[k - 1];
      for (int z = t.opstart[i + 1]; z < t.opstart[i + 2]; ++z) {
        if (t.op_a[z] != ap) continue;
        double s = CDZ_FINF;
        for (int s2 = 0; s2 < t.sig[k - 1]; ++s2) s = fmin2(s, V.E(i + 2, k - 2, t.op_c[z], s2) + d2[s2]);
        best = fmin2(best, t.op_x[z] + g.gtm[P][t.op_b[z]][t.rs_y[r]] + s);
      }
    }
  } else {
    const double* gi = b.GI + (size_t)t.off[k - 1] * S + t.off[l + 2];
    const int Sk = t.sig[k - 1], Sl = t.sig[l + 2];
    for (int z = t.opstart[i + 1]; z < t.opstart[i + 2]; ++z) {
      if (t.op_a[z] != ap) continue;
      for (int w = t.opstart[j - 1]; w < t.opstart[j]; ++w) {
        if (t.op_c[w] != cp) continue;
        double s = CDZ_FINF;
        for (int s2 = 0; s2 < Sk; ++s2) {
          const double el = V.E(i + 2, k - 2, t.op_c[z], s2);
          if (el >= CDZ_FBIG) continue;
          for (int t2 = 0; t2 < Sl; ++t2) s = fmin2(s, el + gi[(size_t)s2 * S + t2] + V.E(l + 2, j - 2, t2, t.op_a[w]));
        }
        best = fmin2(best, t.op_x[z] + t.op_x[w] + g.gtm[P][t.op_b[z]][t.op_b[w]] + s);
      }
    }
  }
  return g.gin[l1 + l2] + best;
}

__global__ void __launch_bounds__(32) mfe_trace_kernel(const Ctx* ctxp, uint8_t* seq, int32_t* pair, MItem* stk, int stack_cap) {
  __shared__ GModel g;
  const Ctx& cx = *ctxp;
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const CModel& cm = *cx.cm;
  load_gmodel(&g, &cm);
  __syncwarp();
  const MV V{t, b, cm, g};
  const int lane = threadIdx.x;
  const int n = t.n, S = t.S, RS = t.RS;
  const int mh1 = cm.min_hairpin + 1, maxint = cm.max_interior;
  int sp = 0;
  for (int k = lane; k < n; k += 32) { seq[k] = 255; pair[k] = -1; }
  __syncwarp();
  const double* QX = b.Qext;
  auto chain = [&](int p, int q, int s, int tend) {
    int cur = s;
    for (int mp = p; mp <= q; ++mp) {
      const int z0 = t.opstart[mp], cnt = t.opstart[mp + 1] - z0;
      const int k = warp_argmin(lane, cnt, [&](int kk) {
        const int z = z0 + kk;
        return t.op_a[z] == cur ? t.op_x[z] + V.E(mp + 1, q, t.op_c[z], tend) : CDZ_FINF;
      });
      const int z = z0 + k;
      if (lane == 0) seq[mp] = t.op_b[z];
      cur = t.op_c[z];
    }
  };
  // ---- exterior --------------------------------------------------------------------------------------------------------------------------------
  int cb = warp_argmin(lane, t.sig[n], [&](int c) { return QX[t.off[n] + c]; });
  int j = n - 1;
  while (j >= 0) {
    const int z0 = t.opstart[j], nops = t.opstart[j + 1] - z0;
    double v1, v2 = CDZ_FINF;
    const int k1 = warp_argmin(lane, nops, [&](int k) {
      const int z = z0 + k;
      return t.op_c[z] == cb ? QX[t.off[j] + t.op_a[z]] + t.op_x[z] : CDZ_FINF;
    }, &v1);
    int nrc = 0;
    for (int r = t.roff[j]; r < t.roff[j + 1]; ++r) nrc += (t.rs_c[r] == cb);
    const int nls = j - mh1 >= 0 ? t.loff[j - mh1 + 1] : 0;
    auto rsel = [&](int rr) { int r = t.roff[j]; for (;; ++r) if (t.rs_c[r] == cb) { if (rr == 0) break; --rr; } return r; };
    int k2 = 0;
    if (nrc > 0 && nls > 0)
      k2 = warp_argmin(lane, nls * nrc, [&](int idx) {
        const int l = idx / nrc, r = rsel(idx % nrc);
        return QX[t.off[t.lspos[l]] + t.ls_a[l]] + b.QB[(size_t)l * RS + r];
      }, &v2);
    if (v1 <= v2) {
      const int z = z0 + k1;
      if (lane == 0) seq[j] = t.op_b[z];
      cb = t.op_a[z];
      j -= 1;
    } else {
      const int l = k2 / nrc, r = rsel(k2 % nrc), k = t.lspos[l];
      if (lane == 0) stk[sp] = MItem{MI_QB, k, j, (short)t.ls_a[l], (short)t.ls_x[l], (short)t.rs_y[r], (short)cb};
      ++sp;
      cb = t.ls_a[l];
      j = k - 1;
    }
  }
  __syncwarp();
  while (sp > 0) {
    --sp;
    const MItem it = stk[sp];
    __syncwarp();
    const int i = it.i;
    j = it.j;
    const int offi = t.off[i], offj1 = t.off[j + 1];
    if (it.type == MI_QM) {
      const double vml = b.QML[(size_t)(offi + it.a) * S + offj1 + it.c];
      const int kb0 = t.off[i + 1];
      const double* A = b.QM + (size_t)(offi + it.a) * S;
      const double* Bt = b.QM1T + (size_t)(offj1 + it.c) * S;
      double v2 = CDZ_FINF;
      int k2 = 0;
      if (offj1 > kb0) k2 = warp_argmin(lane, offj1 - kb0, [&](int k) { return A[kb0 + k] + Bt[kb0 + k]; }, &v2);
      if (vml <= v2) {
        if (lane == 0) stk[sp] = MItem{MI_QML, i, j, it.a, 0, 0, it.c};
        ++sp;
      } else {
        const int kb = kb0 + k2, k = t.bondpos[kb], s = kb - t.off[k];
        if (lane == 0) {
          stk[sp] = MItem{MI_QM, i, k - 1, it.a, 0, 0, (short)s};
          stk[sp + 1] = MItem{MI_QM1, k, j, (short)s, 0, 0, it.c};
        }
        sp += 2;
      }
    } else if (it.type == MI_QML) {
      const int z0 = t.opstart[i], nops = t.opstart[i + 1] - z0;
      const int k = warp_argmin(lane, 1 + nops, [&](int kk) {
        if (kk == 0) return b.QM1T[(size_t)(offj1 + it.c) * S + offi + it.a];
        const int z = z0 + kk - 1;
        if (t.op_a[z] != it.a || i + 1 > j) return CDZ_FINF;
        return g.gb + t.op_x[z] + b.QML[(size_t)(t.off[i + 1] + t.op_c[z]) * S + offj1 + it.c];
      });
      if (k == 0) {
        if (lane == 0) stk[sp] = MItem{MI_QM1, i, j, it.a, 0, 0, it.c};
      } else {
        const int z = z0 + k - 1;
        if (lane == 0) { seq[i] = t.op_b[z]; stk[sp] = MItem{MI_QML, i + 1, j, (short)t.op_c[z], 0, 0, it.c}; }
      }
      ++sp;
    } else if (it.type == MI_QM1) {
      const int z0 = t.opstart[j], nops = t.opstart[j + 1] - z0;
      const int k = warp_argmin(lane, 16 + nops, [&](int kk) {
        if (kk < 16) return V.can(kk >> 2, kk & 3) ? g.gc + V.QB(i, j, it.a, kk >> 2, kk & 3, it.c) : CDZ_FINF;
        const int z = z0 + kk - 16;
        if (t.op_c[z] != it.c || j - 1 < i) return CDZ_FINF;
        return g.gb + b.QM1T[(size_t)(t.off[j] + t.op_a[z]) * S + offi + it.a] + t.op_x[z];
      });
      if (k < 16) {
        if (lane == 0) stk[sp] = MItem{MI_QB, i, j, it.a, (short)(k >> 2), (short)(k & 3), it.c};
      } else {
        const int z = z0 + k - 16;
        if (lane == 0) { seq[j] = t.op_b[z]; stk[sp] = MItem{MI_QM1, i, j - 1, it.a, 0, 0, (short)t.op_a[z]}; }
      }
      ++sp;
    } else {
      // ---- QB(i,j,a,x,y,c) -----------------------------------------------------------------------------------------------------------------
      const int x = it.x, y = it.y, d = j - i, P = V.pt(x, y);
      if (lane == 0) { seq[i] = (uint8_t)x; seq[j] = (uint8_t)y; pair[i] = j; pair[j] = i; }
      const int zi0 = t.opstart[i], ni = t.opstart[i + 1] - zi0, zj0 = t.opstart[j], nj = t.opstart[j + 1] - zj0;
      const int npz = ni * nj;
      auto zw = [&](int pz, int& ap, int& cp) {
        const int zi = zi0 + pz / nj, zj = zj0 + pz % nj;
        ap = t.op_c[zi]; cp = t.op_a[zj];
        if (t.op_a[zi] != it.a || t.op_b[zi] != x || t.op_b[zj] != y || t.op_c[zj] != it.c) return CDZ_FINF;
        return t.op_x[zi] + t.op_x[zj];
      };
      const int p = i + 1, q = j - 1;
      const double gh = -log(t.wh[d - 1]);
      const int zp0 = t.opstart[p], np = t.opstart[p + 1] - zp0, zq0 = t.opstart[q], nq = t.opstart[q + 1] - zq0;
      // hairpin: per compatible (z_i, z_j) the smallest (z_p, z_q); the pair of loop-end operators is resolved after the choice
      auto hp_ends = [&](int ap, int cp, int kk) {
        const int zp = zp0 + kk / nq, zq = zq0 + kk % nq;
        if (t.op_a[zp] != ap || t.op_c[zq] != cp) return CDZ_FINF;
        return t.op_x[zp] + t.op_x[zq] + V.E(p + 1, q - 1, t.op_c[zp], t.op_a[zq]) + g.gtm[P][t.op_b[zp]][t.op_b[zq]];
      };
      double vh;
      const int kh = warp_argmin(lane, npz, [&](int pz) {
        int ap, cp;
        const double w0 = zw(pz, ap, cp);
        if (w0 >= CDZ_FBIG) return CDZ_FINF;
        double best = CDZ_FINF;
        for (int kk = 0; kk < np * nq; ++kk) best = fmin2(best, hp_ends(ap, cp, kk));
        return w0 + gh + best;
      }, &vh);
      // one inner pair: terms numbered by total size, then l1; (z_i, z_j) inner
      const int tmax = min(maxint, d - 2 - mh1);
      const int nterm = tmax >= 0 ? (tmax + 1) * (tmax + 2) / 2 : 0;
      auto term_l1l2 = [&](int term, int& l1, int& l2) {
        int tt = (int)((sqrt(8.0 * term + 1.0) - 1.0) * 0.5);
        while ((tt + 1) * (tt + 2) / 2 <= term) ++tt;
        while (tt * (tt + 1) / 2 > term) --tt;
        l1 = term - tt * (tt + 1) / 2;
        l2 = tt - l1;
      };
      double vl = CDZ_FINF;
      int kl = 0;
      if (nterm > 0)
        kl = warp_argmin(lane, nterm * npz, [&](int idx) {
          int ap, cp, l1, l2;
          const double w0 = zw(idx % npz, ap, cp);
          if (w0 >= CDZ_FBIG) return CDZ_FINF;
          term_l1l2(idx / npz, l1, l2);
          return w0 + mfe_loop_value(V, i, j, p + l1, q - l2, P, ap, cp);
        }, &vl);
      // multiloop: (z_i, z_j) x split bond
      const int kb0 = t.off[i + 2], kb1 = t.off[j];
      const int nml = kb1 > kb0 ? kb1 - kb0 : 0;
      double vm = CDZ_FINF;
      int km = 0;
      if (nml > 0)
        km = warp_argmin(lane, npz * nml, [&](int idx) {
          int ap, cp;
          const double w0 = zw(idx / nml, ap, cp);
          if (w0 >= CDZ_FBIG) return CDZ_FINF;
          const int kb = kb0 + idx % nml;
          return w0 + g.ga_c + b.QM[(size_t)(t.off[p] + ap) * S + kb] + b.QM1T[(size_t)(t.off[q + 1] + cp) * S + kb];
        }, &vm);
      int ap, cp;
      if (vh <= vl && vh <= vm) {
        zw(kh, ap, cp);
        const int ke = warp_argmin(lane, np * nq, [&](int kk) { return hp_ends(ap, cp, kk); });
        const int zp = zp0 + ke / nq, zq = zq0 + ke % nq;
        if (lane == 0) { seq[p] = t.op_b[zp]; seq[q] = t.op_b[zq]; }
        chain(p + 1, q - 1, t.op_c[zp], t.op_a[zq]);
      } else if (vm <= vl) {
        zw(km / nml, ap, cp);
        const int kb = kb0 + km % nml, k = t.bondpos[kb], s = kb - t.off[k];
        if (lane == 0) {
          stk[sp] = MItem{MI_QM, p, k - 1, (short)ap, 0, 0, (short)s};
          stk[sp + 1] = MItem{MI_QM1, k, q, (short)s, 0, 0, (short)cp};
        }
        sp += 2;
      } else {
        int l1, l2;
        zw(kl % npz, ap, cp);
        term_l1l2(kl / npz, l1, l2);
        const int k = p + l1, l = q - l2;
        // level B: (left side operators) x (right side operators) x (x', y')
        const int n1 = l1 == 0 ? 1 : t.opstart[i + 2] - t.opstart[i + 1], n2 = l1 >= 2 ? t.opstart[k] - t.opstart[k - 1] : 1;
        const int n3 = l2 >= 2 ? t.opstart[l + 2] - t.opstart[l + 1] : 1, n4 = l2 == 0 ? 1 : t.opstart[j] - t.opstart[j - 1];
        auto decode = [&](int f, int& z1, int& z2, int& z3, int& z4, int& xp, int& yp) {
          xp = (f >> 2) & 3; yp = f & 3; f >>= 4;
          z4 = t.opstart[j - 1] + f % n4; f /= n4;
          z3 = t.opstart[l + 1] + f % n3; f /= n3;
          z2 = t.opstart[k - 1] + f % n2; f /= n2;
          z1 = t.opstart[i + 1] + f;
        };
        auto side = [&](int f, int& s_, int& tb_) {
          int z1, z2, z3, z4, xp, yp;
          decode(f, z1, z2, z3, z4, xp, yp);
          if (!V.can(xp, yp)) return CDZ_FINF;
          int u = 0, up = 0, v = 0, vp = 0;
          double w = 0.0;
          s_ = ap; tb_ = cp;
          if (l1 == 1) { if (t.op_a[z1] != ap) return CDZ_FINF; u = up = t.op_b[z1]; s_ = t.op_c[z1]; w += t.op_x[z1]; }
          else if (l1 >= 2) {
            if (t.op_a[z1] != ap) return CDZ_FINF;
            u = t.op_b[z1]; up = t.op_b[z2]; s_ = t.op_c[z2];
            w += t.op_x[z1] + V.E(i + 2, k - 2, t.op_c[z1], t.op_a[z2]) + t.op_x[z2];
          }
          if (l2 == 1) { if (t.op_c[z4] != cp) return CDZ_FINF; v = vp = t.op_b[z4]; tb_ = t.op_a[z4]; w += t.op_x[z4]; }
          else if (l2 >= 2) {
            if (t.op_c[z4] != cp) return CDZ_FINF;
            vp = t.op_b[z3]; v = t.op_b[z4]; tb_ = t.op_a[z3];
            w += t.op_x[z3] + V.E(l + 2, j - 2, t.op_c[z3], t.op_a[z4]) + t.op_x[z4];
          }
          double e;
          if (l1 == 0 && l2 == 0) e = g.gst[P][V.pt(xp, yp)];
          else if (l1 == 0 || l2 == 0) e = g.gbu[l1 + l2] + (l1 + l2 == 1 ? g.gst[P][V.pt(xp, yp)] : 0.0);
          else e = g.gin[l1 + l2] + g.gtm[P][u][v] + g.gtm[V.pt(yp, xp)][vp][up];
          return w + e + V.QB(k, l, s_, xp, yp, tb_);
        };
        const int f = warp_argmin(lane, n1 * n2 * n3 * n4 * 16, [&](int ff) { int s_, tb_; return side(ff, s_, tb_); });
        int z1, z2, z3, z4, xp, yp, s_, tb_;
        decode(f, z1, z2, z3, z4, xp, yp);
        side(f, s_, tb_);
        if (l1 >= 1 && lane == 0) seq[i + 1] = t.op_b[z1];
        if (l1 >= 2) {
          if (lane == 0) seq[k - 1] = t.op_b[z2];
          chain(i + 2, k - 2, t.op_c[z1], t.op_a[z2]);
        }
        if (l2 >= 1 && lane == 0) seq[j - 1] = t.op_b[z4];
        if (l2 >= 2) {
          if (lane == 0) seq[l + 1] = t.op_b[z3];
          chain(l + 2, j - 2, t.op_c[z3], t.op_a[z4]);
        }
        if (lane == 0) stk[sp] = MItem{MI_QB, k, l, (short)s_, (short)xp, (short)yp, (short)tb_};
        ++sp;
      }
    }
    __syncwarp();
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------------------------------------------
int cdz_make_tables(const cdz_model* m, const cdz_tt* tt, int precision, void* ws, size_t ws_bytes, cudaStream_t st, cdz_tables** out);

extern "C" int cdz_mfe(const cdz_model* m, const cdz_tt* tt, void* workspace_dev, size_t workspace_bytes, void* stream,
                       double* fmin_host, uint8_t* seq_dev, int32_t* pair_dev) {
  if (!m || !tt || !fmin_host || ((seq_dev == nullptr) != (pair_dev == nullptr))) {
    cdz_set_error("cdz_mfe: bad argument (model, tensor train and fmin_host are required; seq_dev and pair_dev go together)");
    return CDZ_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  cdz_tables* T = nullptr;
  int rc = cdz_make_tables(m, tt, CDZ_FP64, workspace_dev, workspace_bytes, st, &T);
  if (rc != CDZ_OK) return rc;
  const int n = tt->n;
  mfe_init_kernel<<<148 * 8, 256, 0, st>>>(T->d_ctx);
  mfe_init2_kernel<<<148, 256, 0, st>>>(T->d_ctx);
  const MPlan pl = mplan(tt->MS, tt->maxL, tt->maxR, m->c.nps);
  const size_t smem = sizeof(double) * pl.total;
  cudaError_t e = cudaFuncSetAttribute(mfe_cell_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  for (int d = 0; d < n && e == cudaSuccess; ++d) mfe_cell_kernel<<<(unsigned)(n - d), MT, smem, st>>>(T->d_ctx, d, tt->maxL, tt->maxR);
  mfe_ext_kernel<<<1, 1024, 0, st>>>(T->d_ctx);
  MItem* stack = nullptr;
  if (seq_dev && e == cudaSuccess) {
    const int cap = n / 2 + 16;
    e = cudaMallocAsync((void**)&stack, sizeof(MItem) * (size_t)cap, st);
    if (e == cudaSuccess) mfe_trace_kernel<<<1, 32, 0, st>>>(T->d_ctx, seq_dev, pair_dev, stack, cap);
  }
  double f = 0.0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&f, T->h.tab.result, sizeof(double), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && stack) e = cudaFreeAsync(stack, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  cdz_tables_destroy(T);
  if (e != cudaSuccess) { cdz_set_error(std::string("cdz_mfe: ") + cudaGetErrorString(e)); return CDZ_ECUDA; }
  *fmin_host = f;
  return CDZ_OK;
}
