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
//   2. block_kernel  : one CTA per block walks the in-block anti-diagonals (one warp per cell): closed cells Qb
//                      (hairpin, stack, bulge, interior <= 30, multiloop closure), Qm1 / Qml rank updates and the
//                      two in-block edge ranges of the split sum,
//   3. at D = 1,2,4,..: plan_kernel + rescale_kernel re-centre the per-position power-of-two scales (a-7).
// ext_kernel then runs the exterior recursion block column by block column.
#include <math.h>

#include <algorithm>

#include "cdz_internal.h"

namespace {

// (l1,l2) with l1,l2 >= 2 sorted by l1+l2 (then l1): terms with total <= t form a prefix of length (t-3)(t-2)/2
__constant__ uint8_t c_l1[384];
__constant__ uint8_t c_l2[384];

struct Cell {
  const DevTT& t;
  const DevTab& b;
  const CModel& m;
  int lane;
  __device__ Cell(const DevTT& t_, const DevTab& b_, const CModel& m_, int lane_) : t(t_), b(b_), m(m_), lane(lane_) {}
};

__device__ __forceinline__ int pow2ceil(int v) {
  int p = 1;
  while (p < v) p <<= 1;
  return p;
}

// out[e] = sum_t term(e,t) for e < nE, t < nT: lanes split entries x term slices, shuffle-reduce the slices
template <typename F>
__device__ __forceinline__ void warp_terms(int lane, int nE, int nT, double* out, F term) {
  for (int e0 = 0; e0 < nE; e0 += 32) {
    const int rem = nE - e0;
    const int width = rem >= 32 ? 32 : pow2ceil(rem);
    const int e = e0 + (lane & (width - 1));
    const int ts = lane / width, nts = 32 / width;
    double acc = 0.0;
    if (e < nE)
      for (int tt = ts; tt < nT; tt += nts) acc += term(e, tt);
    for (int o = width; o < 32; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (ts == 0 && e < nE) out[e] = acc;
  }
  __syncwarp();
}

// E(p,q)[a][c] = (Tbar_p .. Tbar_q)[a][c]; identity when q == p-1
__device__ __forceinline__ double Eval(const DevTT& t, const DevTab& b, int p, int q, int a, int c) {
  if (q < p) return a == c ? 1.0 : 0.0;
  return b.EM[(size_t)(t.off[p] + a) * t.S + t.off[q + 1] + c];
}

__device__ __forceinline__ int find_l(const DevTT& t, int pos, int a, int x) {
  for (int l = t.loff[pos]; l < t.loff[pos + 1]; ++l)
    if (t.ls_a[l] == a && t.ls_x[l] == x) return l - t.loff[pos];
  return -1;
}
__device__ __forceinline__ int find_r(const DevTT& t, int pos, int y, int c) {
  for (int r = t.roff[pos]; r < t.roff[pos + 1]; ++r)
    if (t.rs_y[r] == y && t.rs_c[r] == c) return r - t.roff[pos];
  return -1;
}

struct Scratch {
  double *B, *XE, *Z1, *Z2, *Y, *SB, *IN, *QBc, *V1, *V2;
};

__host__ __device__ inline int scratch_doubles(int MS, int nps, int maxL, int maxR) {
  return 2 * MS * MS + maxL * MS + MS * maxR + 2 * maxL * maxR + 2 * nps * MS * MS + 2 * MS * MS;
}

__device__ __forceinline__ Scratch carve_scratch(double* s, int MS, int nps, int maxL, int maxR) {
  Scratch k;
  k.B = s; s += MS * MS;
  k.XE = s; s += MS * MS;
  k.Z1 = s; s += maxL * MS;
  k.Z2 = s; s += MS * maxR;
  k.Y = s; s += maxL * maxR;
  k.QBc = s; s += maxL * maxR;
  k.SB = s; s += nps * MS * MS;
  k.IN = s; s += nps * MS * MS;
  k.V1 = s; s += MS * MS;
  k.V2 = s; s += MS * MS;
  return k;
}

// ------------------------------------------------------------------------------------------------
// one cell (i,j); kb_lo..kb_hi: bond-index range of the split sum handled here (v1: the whole range)
// ------------------------------------------------------------------------------------------------
// side stretch ES(p,len)[a][c] = (Tbar_p .. Tbar_{p+len-1})[a][c], row stride MS
__device__ __forceinline__ const double* ESp(const DevTT& t, const DevTab& b, int p, int len) {
  return b.ES + ((size_t)p * 31 + len) * (t.MS * t.MS);
}

constexpr int XU = 27;  // interior-loop totals u = l1 + l2 = 4 .. 30 with l1, l2 >= 2

// xs: shared-memory state of column j: X_u(i,j)[a2][c2] at xs[((u-4)*MS + a2)*Sc + c2], the bond-only body
// sum_{l1+l2=u} E(i+2,k-2) Gi(k,l) E(l+2,j-2) of SURVEY App. A.5 (unweighted); bottom: first row of an off-diagonal block
__device__ void compute_cell(const DevTT& t, const DevTab& b, const CModel& m, const Scratch& sc, int lane, int i,
                             int j, int I, int J, int nsplit, double* xs, bool bottom) {
  const int n = t.n, S = t.S, RS = t.RS, MS = t.MS;
  const int d = j - i;
  const int Si = t.sig[i], Sj1 = t.sig[j + 1];
  const int offi = t.off[i], offj1 = t.off[j + 1];
  const int nLi = t.loff[i + 1] - t.loff[i], nRj = t.roff[j + 1] - t.roff[j];
  const int mh1 = m.min_hairpin + 1;  // smallest d of a closed cell
  const int maxint = m.max_interior;
  const int nps = m.nps;

  // ---- E(i,j) = E(i,j-1) Tbar_j -------------------------------------------------------------------
  {
    const int Sj = t.sig[j];
    for (int e = lane; e < Si * Sj1; e += 32) {
      const int a = e / Sj1, c = e % Sj1;
      double v = 0.0;
      for (int s = 0; s < Sj; ++s) v += Eval(t, b, i, j - 1, a, s) * t.Tbar[((size_t)j * MS + s) * MS + c];
      b.EM[(size_t)(offi + a) * S + offj1 + c] = v;
    }
  }

  // ---- X_u(i,j), u = 4..30: direct sum on the first row of an off-diagonal block, else the row recursion
  //      X_u(i,j) = Tbar_{i+2} X_{u-1}(i+1,j) + Gi(i+3, j+1-u) E(j+3-u, j-2)   (l1 >= 3 terms | l1 = 2 term)
  if (d >= 4) {
    const int Sa = t.sig[i + 2], Sc = t.sig[j - 1];
    const int nX = XU * Sa * Sc;
    if (bottom) {
      for (int e = lane; e < nX; e += 32) {
        const int c2 = e % Sc, a2 = (e / Sc) % Sa, u = 4 + e / (Sc * Sa);
        double acc = 0.0;
        for (int l1 = 2; l1 <= u - 2; ++l1) {
          const int l2 = u - l1, rp = i + l1, cp = j + 1 - l2;  // Gi(k,l) sits at row position k-1, column position l+2
          if (cp - rp - 3 < mh1) continue;                       // inner span l - k
          const int Sk = t.sig[rp], Sl = t.sig[cp];
          const double* EL = ESp(t, b, i + 2, l1 - 2) + a2 * MS;
          const double* ER = ESp(t, b, cp, l2 - 2) + c2;
          const double* g = b.GI + (size_t)t.off[rp] * S + t.off[cp];
          for (int s2 = 0; s2 < Sk; ++s2) {
            const double el = EL[s2];
            if (el == 0.0) continue;
            double r = 0.0;
            for (int u2 = 0; u2 < Sl; ++u2) r += g[(size_t)s2 * S + u2] * ER[u2 * MS];
            acc += el * r;
          }
        }
        xs[((u - 4) * MS + a2) * Sc + c2] = acc;
      }
      __syncwarp();
    } else {
      const int Sa3 = t.sig[i + 3];
      const double* Tb = t.Tbar + (size_t)(i + 2) * MS * MS;
      // in place, descending element order: element (u,..) reads old elements of u-1 only
      for (int hi = nX; hi > 0; hi -= 64) {
        double val[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
          const int e = hi - 1 - (r * 32 + lane);
          val[r] = 0.0;
          if (e < 0) continue;
          const int c2 = e % Sc, a2 = (e / Sc) % Sa, u = 4 + e / (Sc * Sa);
          double acc = 0.0;
          if (u > 4)
            for (int a3 = 0; a3 < Sa3; ++a3) acc += Tb[a2 * MS + a3] * xs[((u - 5) * MS + a3) * Sc + c2];
          const int cp = j + 3 - u;
          if (cp - (i + 2) - 3 >= mh1) {
            const int Sl = t.sig[cp];
            const double* g = b.GI + (size_t)(t.off[i + 2] + a2) * S + t.off[cp];
            const double* ER = ESp(t, b, cp, u - 4) + c2;
            for (int u2 = 0; u2 < Sl; ++u2) acc += g[u2] * ER[u2 * MS];
          }
          val[r] = acc;
        }
        __syncwarp();
#pragma unroll
        for (int r = 0; r < 2; ++r) {
          const int e = hi - 1 - (r * 32 + lane);
          if (e < 0) continue;
          const int c2 = e % Sc, a2 = (e / Sc) % Sa, u = 4 + e / (Sc * Sa);
          xs[((u - 4) * MS + a2) * Sc + c2] = val[r];
        }
        __syncwarp();
      }
    }
  }

  if (d >= mh1) {
    const int p = i + 1, q = j - 1;
    const int S1 = t.sig[p], S2 = t.sig[j];         // a' in Sigma_{i+1}, c' in Sigma_j
    const int Sp1 = t.sig[p + 1], Sq = t.sig[q];    // a'' in Sigma_{p+1}, c'' in Sigma_q
    const int nLp = t.loff[p + 1] - t.loff[p], nRq = t.roff[q + 1] - t.roff[q];
    const int loffp = t.loff[p], roffq = t.roff[q];
    const int opp0 = t.opstart[p], opp1 = t.opstart[p + 1], opq0 = t.opstart[q], opq1 = t.opstart[q + 1];
    const int span = q - p;

    // ---- XE = sum_u win[u] X_u + hairpin interior (X_u state updated above) -----------------------------------
    {
      warp_terms(lane, Sp1 * Sq, XU, sc.XE, [&](int e, int tt) {
        const int a2 = e / Sq, c2 = e % Sq;
        return tt + 4 <= maxint ? m.win[tt + 4] * xs[(tt * MS + a2) * Sq + c2] : 0.0;
      });
      const double wh = t.wh[d - 1];
      for (int e = lane; e < Sp1 * Sq; e += 32) sc.XE[e] += wh * Eval(t, b, p + 1, q - 1, e / Sq, e % Sq);
      __syncwarp();
    }
    // ---- B: pair-independent bond body: multiloop closure + bulges of size >= 2 ------------------------
    warp_terms(lane, S1 * S2, 59, sc.B, [&](int e, int tt) {
      const int a1 = e / S2, c1 = e % S2;
      if (tt == 0) return m.wac * b.M2[(size_t)(t.off[p] + a1) * S + t.off[q + 1] + c1];
      if (tt < 30) {  // left bulge, l1 = tt+1
        const int l1 = tt + 1, k = p + l1;
        if (l1 > maxint || q - k < mh1) return 0.0;
        const int Sk = t.sig[k];
        const double* EL = ESp(t, b, p, l1) + a1 * MS;
        double sum = 0.0;
        for (int s = 0; s < Sk; ++s) sum += EL[s] * b.QBS[(size_t)(t.off[k] + s) * S + t.off[q + 1] + c1];
        return m.wbu[l1] * sum;
      }
      const int l2 = tt - 28, l = q - l2;  // right bulge
      if (l2 > maxint || l - p < mh1) return 0.0;
      const int Sl = t.sig[l + 1];
      const double* ER = ESp(t, b, l + 1, l2) + c1;
      double sum = 0.0;
      for (int u = 0; u < Sl; ++u) sum += b.QBS[(size_t)(t.off[p] + a1) * S + t.off[l + 1] + u] * ER[u * MS];
      return m.wbu[l2] * sum;
    });
    // ---- Z1: l1 = 1, l2 >= 2 ------------------------------------------------------------------------
    warp_terms(lane, nLp * Sq, 28, sc.Z1, [&](int e, int tt) {
      const int lst = e / Sq, c2 = e % Sq;
      const int l2 = tt + 2, l = q - l2;
      if (1 + l2 > maxint || l - (p + 1) < mh1) return 0.0;
      const int Sl = t.sig[l + 2];
      const double* dd = b.D1 + (size_t)(loffp + lst) * S + t.off[l + 2];
      const double* ER = ESp(t, b, l + 2, l2 - 2) + c2;
      double sum = 0.0;
      for (int u = 0; u < Sl; ++u) sum += dd[u] * ER[u * MS];
      return m.win[1 + l2] * sum;
    });
    // ---- Z2: l2 = 1, l1 >= 2 ------------------------------------------------------------------------
    warp_terms(lane, Sp1 * nRq, 28, sc.Z2, [&](int e, int tt) {
      const int a2 = e / nRq, r = e % nRq;
      const int l1 = tt + 2, k = p + l1;
      if (l1 + 1 > maxint || (q - 1) - k < mh1) return 0.0;
      const int Sk = t.sig[k - 1];
      const double* EL = ESp(t, b, p + 1, l1 - 2) + a2 * MS;
      double sum = 0.0;
      for (int s = 0; s < Sk; ++s) sum += EL[s] * b.D2[(size_t)(t.off[k - 1] + s) * RS + roffq + r];
      return m.win[l1 + 1] * sum;
    });
    // ---- Y[(a',u),(v,c')]: everything that carries the closing mismatch tmm[p(x,y)][u][v] -----------------
    {
      const bool v11 = (2 <= maxint) && ((q - 1) - (p + 1) >= mh1);
      for (int e = lane; e < nLp * nRq; e += 32) {
        const int lst = e / nRq, r = e % nRq;
        double y = v11 ? m.win[2] * b.DD[(size_t)(loffp + lst) * RS + roffq + r] : 0.0;
        for (int z = opp0; z < opp1; ++z) {
          if (t.op_l[z] != lst) continue;
          const double xz = t.op_x[z];
          const int cz = t.op_c[z];
          y += xz * sc.Z2[cz * nRq + r];
          for (int w = opq0; w < opq1; ++w)
            if (t.op_r[w] == r) y += xz * t.op_x[w] * sc.XE[cz * Sq + t.op_a[w]];
        }
        for (int w = opq0; w < opq1; ++w)
          if (t.op_r[w] == r) y += t.op_x[w] * sc.Z1[lst * Sq + t.op_a[w]];
        sc.Y[e] = y;
      }
      __syncwarp();
    }
    // ---- SB[a'][slot'][c']: inner pair identity kept (stack, bulges of size 1) --------------------------
    {
      const bool vst = span >= mh1, vbl = (1 <= maxint) && (q - (p + 1) >= mh1);
      for (int e = lane; e < S1 * nps * S2; e += 32) {
        const int c1 = e % S2, sl = (e / S2) % nps, a1 = e / (S2 * nps);
        const int xp = m.slot_x[sl], yp = m.slot_y[sl];
        double v = 0.0;
        const int lst = find_l(t, p, a1, xp), r = find_r(t, q, yp, c1);
        if (vst && lst >= 0 && r >= 0) v += b.QB[(size_t)(loffp + lst) * RS + roffq + r];
        if (vbl) {
          double s1 = 0.0, s2 = 0.0;
          if (r >= 0)
            for (int l2 = t.loff[p + 1]; l2 < t.loff[p + 2]; ++l2)
              if (t.ls_x[l2] == xp)
                s1 += t.Tbar[((size_t)p * MS + a1) * MS + t.ls_a[l2]] * b.QB[(size_t)l2 * RS + roffq + r];
          if (lst >= 0)
            for (int r2 = t.roff[q - 1]; r2 < t.roff[q]; ++r2)
              if (t.rs_y[r2] == yp)
                s2 += b.QB[(size_t)(loffp + lst) * RS + r2] * t.Tbar[((size_t)q * MS + t.rs_c[r2]) * MS + c1];
          v += m.wbu[1] * (s1 + s2);
        }
        sc.SB[e] = v;
      }
      __syncwarp();
    }
    // ---- inner[slot][a'][c'] -----------------------------------------------------------------------------
    for (int e = lane; e < nps * S1 * S2; e += 32) {
      const int c1 = e % S2, a1 = (e / S2) % S1, sl = e / (S2 * S1);
      const int P = m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]];
      double v = sc.B[a1 * S2 + c1];
      for (int lst = 0; lst < nLp; ++lst) {
        if (t.ls_a[loffp + lst] != a1) continue;
        const int u = t.ls_x[loffp + lst];
        for (int r = 0; r < nRq; ++r)
          if (t.rs_c[roffq + r] == c1) v += m.wtm[P][u][t.rs_y[roffq + r]] * sc.Y[lst * nRq + r];
      }
      for (int s2 = 0; s2 < nps; ++s2)
        v += m.wst[P][m.ptype[m.slot_x[s2] * 4 + m.slot_y[s2]]] * sc.SB[(a1 * nps + s2) * S2 + c1];
      sc.IN[e] = v;
    }
    __syncwarp();
    // ---- Qb[(a,x),(y,c)] = can(x,y) sum T_i[a,x,a'] T_j[c',y,c] inner -------------------------------------
    {
      const int opi0 = t.opstart[i], opi1 = t.opstart[i + 1], opj0 = t.opstart[j], opj1 = t.opstart[j + 1];
      for (int e = lane; e < nLi * nRj; e += 32) {
        const int lst = e / nRj, r = e % nRj;
        const int sl = m.pslot[t.ls_x[t.loff[i] + lst] * 4 + t.rs_y[t.roff[j] + r]];
        double v = 0.0;
        if (sl >= 0)
          for (int z = opi0; z < opi1; ++z) {
            if (t.op_l[z] != lst) continue;
            for (int w = opj0; w < opj1; ++w)
              if (t.op_r[w] == r) v += t.op_x[z] * t.op_x[w] * sc.IN[(sl * S1 + t.op_c[z]) * S2 + t.op_a[w]];
          }
        sc.QBc[e] = v;
        b.QB[(size_t)(t.loff[i] + lst) * RS + t.roff[j] + r] = v;
      }
      __syncwarp();
    }
  } else {
    for (int e = lane; e < nLi * nRj; e += 32) {
      sc.QBc[e] = 0.0;
      b.QB[(size_t)(t.loff[i] + e / nRj) * RS + t.roff[j] + e % nRj] = 0.0;
    }
    __syncwarp();
  }

  // ---- Qbs, Qm1, Qml ------------------------------------------------------------------------------------
  for (int e = lane; e < Si * Sj1; e += 32) {
    const int a = e / Sj1, c = e % Sj1;
    double qbs = 0.0;
    for (int lst = 0; lst < nLi; ++lst)
      if (t.ls_a[t.loff[i] + lst] == a)
        for (int r = 0; r < nRj; ++r)
          if (t.rs_c[t.roff[j] + r] == c) qbs += sc.QBc[lst * nRj + r];
    double qm1 = m.wc * qbs;
    if (j - 1 >= i) {
      const int Sj = t.sig[j];
      double s1 = 0.0;
      for (int s = 0; s < Sj; ++s)
        s1 += b.QM1T[(size_t)(t.off[j] + s) * S + offi + a] * t.Tbar[((size_t)j * MS + s) * MS + c];
      qm1 += m.wb * s1;
    }
    double qml = qm1;
    if (i + 1 <= j) {
      const int Si1 = t.sig[i + 1];
      double s1 = 0.0;
      for (int s = 0; s < Si1; ++s)
        s1 += t.Tbar[((size_t)i * MS + a) * MS + s] * b.QML[(size_t)(t.off[i + 1] + s) * S + offj1 + c];
      qml += m.wb * s1;
    }
    b.QBS[(size_t)(offi + a) * S + offj1 + c] = qbs;
    b.QM1T[(size_t)(offj1 + c) * S + offi + a] = qm1;
    b.QML[(size_t)(offi + a) * S + offj1 + c] = qml;
    sc.V1[e] = qml;
  }
  __syncwarp();

  // ---- M2(i,j) = sum_k Qm(i,k-1) Qm1(k,j); Qm = Qml + M2 --------------------------------------------------
  // blocks I < K < J: partial tiles of gemm_kernel, summed in split order; then the bonds of positions
  // k > i inside block I and k <= j inside block J as contiguous-row dot products
  {
    int ra0, ra1, rb0 = 0, rb1 = 0;
    if (I == J) {
      ra0 = t.off[i + 1];
      ra1 = offj1;
    } else {
      ra1 = (I + 1) * CDZ_TB;
      ra0 = t.posblk[i + 1] == I ? t.off[i + 1] : ra1;
      rb0 = J * CDZ_TB;
      rb1 = offj1;
    }
    const double* gp = b.GP + (size_t)I * nsplit * (CDZ_TB * CDZ_TB) + (size_t)(offi - I * CDZ_TB) * CDZ_TB +
                       (offj1 - J * CDZ_TB);
    for (int e = 0; e < Si * Sj1; ++e) {
      const int a = e / Sj1, c = e % Sj1;
      const double* A = b.QM + (size_t)(offi + a) * S;
      const double* Bt = b.QM1T + (size_t)(offj1 + c) * S;
      double acc = 0.0;
      for (int kb = ra0 + lane; kb < ra1; kb += 32) acc += A[kb] * Bt[kb];
      for (int kb = rb0 + lane; kb < rb1; kb += 32) acc += A[kb] * Bt[kb];
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      for (int sp = 0; sp < nsplit; ++sp) acc += gp[(size_t)sp * (CDZ_TB * CDZ_TB) + a * CDZ_TB + c];
      const double qm = sc.V1[e] + acc;
      if (lane == 0) {
        b.M2[(size_t)(offi + a) * S + offj1 + c] = acc;
        b.QM[(size_t)(offi + a) * S + offj1 + c] = qm;
      }
    }
  }

  // ---- mismatch-dressed extension of Qb(i,j) to [i-1..j+1] (stored at cell (i-1,j+1)) ----------------------
  if (d >= mh1 && i >= 1 && j <= n - 2 && maxint >= 2) {
    const int pi = i - 1, pj = j + 1;
    const int nL2 = t.loff[pi + 1] - t.loff[pi], nR2 = t.roff[pj + 1] - t.roff[pj];
    const int o0 = t.opstart[pi], o1 = t.opstart[pi + 1], w0 = t.opstart[pj], w1 = t.opstart[pj + 1];
    for (int e = lane; e < nL2 * nR2; e += 32) {
      const int lst = e / nR2, r = e % nR2;
      const int up = t.ls_x[t.loff[pi] + lst], vp = t.rs_y[t.roff[pj] + r];
      double v = 0.0;
      for (int z = o0; z < o1; ++z) {
        if (t.op_l[z] != lst) continue;
        for (int w = w0; w < w1; ++w) {
          if (t.op_r[w] != r) continue;
          const int s = t.op_c[z], u = t.op_a[w];
          double in = 0.0;
          for (int l2 = 0; l2 < nLi; ++l2) {
            if (t.ls_a[t.loff[i] + l2] != s) continue;
            const int x = t.ls_x[t.loff[i] + l2];
            for (int r2 = 0; r2 < nRj; ++r2) {
              if (t.rs_c[t.roff[j] + r2] != u) continue;
              const int y = t.rs_y[t.roff[j] + r2];
              if (m.pslot[x * 4 + y] < 0) continue;
              in += m.wtm[m.ptype[y * 4 + x]][vp][up] * sc.QBc[l2 * nRj + r2];
            }
          }
          v += t.op_x[z] * t.op_x[w] * in;
        }
      }
      sc.Y[e] = v;
      b.DD[(size_t)(t.loff[pi] + lst) * RS + t.roff[pj] + r] = v;
    }
    __syncwarp();
    const int Sa = t.sig[pi], Sc = t.sig[pj + 1];
    for (int e = lane; e < Sa * Sc; e += 32) {  // GI
      const int a = e / Sc, c = e % Sc;
      double v = 0.0;
      for (int lst = 0; lst < nL2; ++lst)
        if (t.ls_a[t.loff[pi] + lst] == a)
          for (int r = 0; r < nR2; ++r)
            if (t.rs_c[t.roff[pj] + r] == c) v += sc.Y[lst * nR2 + r];
      b.GI[(size_t)(t.off[pi] + a) * S + t.off[pj + 1] + c] = v;
    }
    for (int e = lane; e < nL2 * Sc; e += 32) {  // D1
      const int lst = e / Sc, c = e % Sc;
      double v = 0.0;
      for (int r = 0; r < nR2; ++r)
        if (t.rs_c[t.roff[pj] + r] == c) v += sc.Y[lst * nR2 + r];
      b.D1[(size_t)(t.loff[pi] + lst) * S + t.off[pj + 1] + c] = v;
    }
    for (int e = lane; e < Sa * nR2; e += 32) {  // D2
      const int a = e / nR2, r = e % nR2;
      double v = 0.0;
      for (int lst = 0; lst < nL2; ++lst)
        if (t.ls_a[t.loff[pi] + lst] == a) v += sc.Y[lst * nR2 + r];
      b.D2[(size_t)(t.off[pi] + a) * RS + t.roff[pj] + r] = v;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// block kernel: one CTA per block (I, I+D); in-block anti-diagonals in order, one warp per cell
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(CDZ_WARPS * 32) block_kernel(const Ctx* ctxs, int D, int nsplit, int scr, int xsz) {
  extern __shared__ double smem[];
  __shared__ CModel cm;
  __shared__ int xoff[CDZ_TB + 2];
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const int I = blockIdx.x, J = I + D;
  if (J >= t.NB) return;
  {
    const int* src = (const int*)cx.cm;
    int* dst = (int*)&cm;
    for (int k = threadIdx.x; k < (int)(sizeof(CModel) / 4); k += blockDim.x) dst[k] = src[k];
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const int n = t.n;
  // rows i in [i0,i1), columns j in [j0,j1): bond position j+1 lies in block J
  const int i0 = t.blk_start[I], i1 = min(t.blk_start[I + 1], n);
  const int j0 = max(t.blk_start[J], 1) - 1, j1 = t.blk_start[J + 1] - 1;
  // per-column X_u state (27 * MS * Sigma_{j-1} doubles each), zero = empty body
  double* xstate = smem;
  if (threadIdx.x == 0) {
    int acc = 0;
    for (int j = j0; j < j1; ++j) {
      xoff[j - j0] = acc;
      acc += XU * t.MS * (j >= 1 ? t.sig[j - 1] : 0);
    }
  }
  for (int k = threadIdx.x; k < xsz; k += blockDim.x) xstate[k] = 0.0;
  __syncthreads();
  const Scratch sc = carve_scratch(smem + xsz + (size_t)warp * scr, t.MS, cm.nps, t.maxL, t.maxR);
  const int dmin = max(0, j0 - (i1 - 1)), dmax = (j1 - 1) - i0;
  for (int d = dmin; d <= dmax; ++d) {
    const int ilo = max(i0, j0 - d), ihi = min(i1 - 1, j1 - 1 - d);
    for (int i = ilo + warp; i <= ihi; i += nw)
      compute_cell(t, cx.tab, cm, sc, lane, i, i + d, I, J, nsplit, xstate + xoff[i + d - j0], I != J && i == i1 - 1);
    __syncthreads();
  }
}

// side stretches ES(p,len), len = 0..30, from the (scaled) transfer matrices; one thread per start position
__global__ void __launch_bounds__(128) side_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.y];
  const DevTT& t = cx.tt;
  const int n = t.n, MS = t.MS, M2 = MS * MS;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  double* out = cx.tab.ES + (size_t)p * 31 * M2;
  const int Sp = t.sig[p];
  for (int e = 0; e < M2; ++e) out[e] = (e / MS == e % MS && e / MS < Sp) ? 1.0 : 0.0;
  for (int len = 1; len <= 30; ++len) {
    const double* prev = out + (size_t)(len - 1) * M2;
    double* cur = out + (size_t)len * M2;
    const int pos = p + len - 1;
    if (pos >= n) {
      for (int e = 0; e < M2; ++e) cur[e] = 0.0;
      continue;
    }
    const double* Tb = t.Tbar + (size_t)pos * M2;
    const int Sm = t.sig[pos], Sn = t.sig[pos + 1];
    for (int a = 0; a < MS; ++a)
      for (int c = 0; c < MS; ++c) {
        double v = 0.0;
        if (a < Sp && c < Sn)
          for (int s2 = 0; s2 < Sm; ++s2) v += prev[a * MS + s2] * Tb[s2 * MS + c];
        cur[a * MS + c] = v;
      }
  }
}

// ------------------------------------------------------------------------------------------------
// split-point GEMM: GP[I][split] = QM[I, K-range] * QM1T[J, K-range]^T, 64x64 tile per CTA, fp64 mma.sync m8n8k4
// ------------------------------------------------------------------------------------------------
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

__global__ void __launch_bounds__(GEMM_THREADS) gemm_kernel(const Ctx* ctxs, int D, int nsplit) {
  extern __shared__ double gsm[];
  const Ctx& cx = ctxs[blockIdx.y];
  const int I = blockIdx.x / nsplit, sp = blockIdx.x % nsplit, J = I + D;
  if (J >= cx.tt.NB) return;
  const size_t S = (size_t)cx.tt.S;
  const int nk = D - 1;  // K blocks I+1 .. J-1
  const int kbeg = (I + 1 + (int)((long long)sp * nk / nsplit)) * CDZ_TB;
  const int kend = (I + 1 + (int)((long long)(sp + 1) * nk / nsplit)) * CDZ_TB;
  const double* A = cx.tab.QM + (size_t)I * CDZ_TB * S;
  const double* Bm = cx.tab.QM1T + (size_t)J * CDZ_TB * S;
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
  double* C = cx.tab.GP + ((size_t)I * nsplit + sp) * (CDZ_TB * CDZ_TB);
#pragma unroll
  for (int mi = 0; mi < 4; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) {
      const int r = wm + mi * 8 + (lane >> 2), c = wn + ni * 8 + 2 * (lane & 3);
      *reinterpret_cast<double2*>(C + r * CDZ_TB + c) = make_double2(acc[mi][ni][0], acc[mi][ni][1]);
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
  if (nw <= 0) return;
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
    case 3: tab = b.D2; colsp = 1; break;
    case 4: tab = b.GI; break;
    case 5: tab = b.QBS; break;
    case 6: tab = b.QM; break;
    case 7: tab = b.QML; break;
    case 8: tab = b.M2; break;
    case 9: tab = b.EM; break;
    default: tab = b.QM1T; lower = 1; break;
  }
  const int nrows = rowsp ? t.LS : t.S;
  const size_t ld = colsp ? (size_t)t.RS : (size_t)t.S;
  const int* Erow = rowsp ? b.EL : b.EB;
  const int* Ecol = colsp ? b.ER : b.EB;
  const int n = t.n, NB = t.NB;
  for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
    const int rb = rowsp ? t.posblk[t.lspos[row]] : row / CDZ_TB;
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
  if (threadIdx.x < CDZ_TB) qx[threadIdx.x] = 0.0;
  __syncthreads();
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    const int p0 = t.blk_start[K], p1 = min(t.blk_start[K + 1], n + 1);
    for (int jj = p0; jj < p1; ++jj) {
      const int Sj = t.sig[jj], oj = t.off[jj] - base;
      for (int c = 0; c < Sj; ++c) {
        double v = 0.0;
        if (jj == 0) {
          v = 1.0;
        } else {
          double part = qx[lane] * Dg[lane * (CDZ_TB + 1) + oj + c] + qx[lane + 32] * Dg[(lane + 32) * (CDZ_TB + 1) + oj + c];
          for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
          v = b.R[base + oj + c] + part;
          const int Sp = t.sig[jj - 1], op = t.off[jj - 1];
          for (int s = 0; s < Sp; ++s) {
            const double q = op >= base ? qx[op - base + s] : b.Qext[op + s];
            v += q * t.Tbar[((size_t)(jj - 1) * MS + s) * MS + c];
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
}

__global__ void zero_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.y];
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < cx.tt.S; k += gridDim.x * blockDim.x) cx.tab.R[k] = 0.0;
}

}  // namespace

static void fill_lut() {
  static bool done = false;
  if (done) return;
  uint8_t a[384], bq[384];
  int k = 0;
  for (int tot = 4; tot <= 30; ++tot)
    for (int l1 = 2; l1 <= tot - 2; ++l1) { a[k] = (uint8_t)l1; bq[k] = (uint8_t)(tot - l1); ++k; }
  cudaMemcpyToSymbol(c_l1, a, k);
  cudaMemcpyToSymbol(c_l2, bq, k);
  done = true;
}

int cdz_launch_inside(cdz_tables* const* ts, int B, cudaStream_t st) {
  fill_lut();
  int NBmax = 1, Smax = 0, nrmax = 0, MS = 1, maxL = 1, maxR = 1, nps = 6;
  for (int b = 0; b < B; ++b) {
    const cdz_tt* tt = ts[b]->tt;
    NBmax = std::max(NBmax, tt->NB);
    Smax = std::max(Smax, tt->S);
    nrmax = std::max(nrmax, std::max(tt->S, tt->LS));
    MS = std::max(MS, tt->MS);
    maxL = std::max(maxL, tt->maxL);
    maxR = std::max(maxR, tt->maxR);
    nps = std::max(nps, ts[b]->model->c.nps);
  }
  const Ctx* d_ctxs = ts[0]->d_ctx;
  Ctx* tmp = nullptr;
  if (B > 1) {
    std::vector<Ctx> h(B);
    for (int b = 0; b < B; ++b) h[b] = ts[b]->h;
    CDZ_CUDA(cudaMallocAsync((void**)&tmp, sizeof(Ctx) * B, st));
    CDZ_CUDA(cudaMemcpyAsync(tmp, h.data(), sizeof(Ctx) * B, cudaMemcpyHostToDevice, st));
    CDZ_CUDA(cudaStreamSynchronize(st));
    d_ctxs = tmp;
  }
  const int scr = scratch_doubles(MS, nps, maxL, maxR);
  const int xsz = XU * MS * (CDZ_TB + 2 * MS);
  int nwarps = CDZ_WARPS;
  while (nwarps > 1 && ((size_t)xsz + (size_t)scr * nwarps) * sizeof(double) > 220 * 1024) --nwarps;
  const size_t smem = ((size_t)xsz + (size_t)scr * nwarps) * sizeof(double);
  if (smem > 220 * 1024) { cdz_set_error("block kernel: shared-memory need exceeds 220 KB"); return CDZ_ENOMEM; }
  CDZ_CUDA(cudaFuncSetAttribute(block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  CDZ_CUDA(cudaFuncSetAttribute(gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM));
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
  mark(4, 2);
  init_kernel<<<dim3(32, B), 256, 0, st>>>(d_ctxs);
  int nmax = 0;
  for (int b = 0; b < B; ++b) nmax = std::max(nmax, ts[b]->tt->n);
  side_kernel<<<dim3((nmax + 127) / 128, B), 128, 0, st>>>(d_ctxs);
  int next_event = 1;
  for (int D = 0; D < NBmax; ++D) {
    const int nblk = NBmax - D;
    const int nsplit = cdz_nsplit(NBmax, D, B);
    if (nsplit > 0) {
      mark(0, 1);
      gemm_kernel<<<dim3(nblk * nsplit, B), GEMM_THREADS, GEMM_SMEM, st>>>(d_ctxs, D, nsplit);
    }
    mark(1, 1);
    block_kernel<<<dim3(nblk, B), nwarps * 32, smem, st>>>(d_ctxs, D, nsplit, scr, xsz);
    if (D == next_event && D + 1 < NBmax) {
      next_event *= 2;
      mark(2, 13);
      plan_kernel<<<B, 1024, NBmax * sizeof(double), st>>>(d_ctxs, D);
      const int gx = std::min(nrmax, 148 * 8);
      for (int which = 0; which <= 10; ++which) rescale_kernel<<<dim3(gx, B), 256, 0, st>>>(d_ctxs, which, D);
      side_kernel<<<dim3((nmax + 127) / 128, B), 128, 0, st>>>(d_ctxs);
    }
  }
  mark(3, 1 + NBmax);
  zero_kernel<<<dim3(32, B), 256, 0, st>>>(d_ctxs);
  for (int K = 0; K < NBmax; ++K) {
    const int rem = Smax - (K + 1) * CDZ_TB;
    const int gx = std::max(1, std::min(148, (rem + 511) / 512));
    ext_kernel<<<dim3(gx, B), 256, 0, st>>>(d_ctxs, K);
  }
  mark(7, 0);  // closing event
  CDZ_CUDA(cudaGetLastError());
  if (tmp) CDZ_CUDA(cudaFreeAsync(tmp, st));
  return CDZ_OK;
}
