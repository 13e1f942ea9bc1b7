// cdz_inside.cu -- wavefront inside kernels (sm_100a).
//
// One warp computes one DP cell (i,j) of the current anti-diagonal d = j-i.  Every quantity of the cell
// is a small dense tensor over tensor-train bond indices and boundary nucleotides (eq 3.8,
// lines 203-211); the recursion is DESIGN.md "Recursion".  All tables are
// row-major matrices over the packed bond / boundary-state index spaces, so the
// split-point sum  M2(i,j) = sum_k Qm(i,k-1) Qm1(k,j)  is the paper's flattened product
// Q_{i,k} Q_{j,k}^T (eq 3.5, Alg S4.2): a dot product of two contiguous rows.
#include <math.h>

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
__device__ void compute_cell(const DevTT& t, const DevTab& b, const CModel& m, const Scratch& sc, int lane, int i,
                             int j) {
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

  if (d >= mh1) {
    const int p = i + 1, q = j - 1;
    const int S1 = t.sig[p], S2 = t.sig[j];         // a' in Sigma_{i+1}, c' in Sigma_j
    const int Sp1 = t.sig[p + 1], Sq = t.sig[q];    // a'' in Sigma_{p+1}, c'' in Sigma_q
    const int nLp = t.loff[p + 1] - t.loff[p], nRq = t.roff[q + 1] - t.roff[q];
    const int loffp = t.loff[p], roffq = t.roff[q];
    const int opp0 = t.opstart[p], opp1 = t.opstart[p + 1], opq0 = t.opstart[q], opq1 = t.opstart[q + 1];
    const int span = q - p;

    // ---- X: interior loops with l1,l2 >= 2 on the mismatch-dressed inner cells ----
    {
      int tmax = min(maxint, span - mh1);
      int nT = tmax >= 4 ? (tmax - 3) * (tmax - 2) / 2 : 0;
      warp_terms(lane, Sp1 * Sq, nT, sc.XE, [&](int e, int tt) {
        const int a2 = e / Sq, c2 = e % Sq;
        const int l1 = c_l1[tt], l2 = c_l2[tt];
        const int k = p + l1, l = q - l2;
        const int Sk = t.sig[k - 1], Sl = t.sig[l + 2];
        const double* g = b.GI + (size_t)t.off[k - 1] * S + t.off[l + 2];
        double sum = 0.0;
        for (int s = 0; s < Sk; ++s) {
          const double el = Eval(t, b, p + 1, k - 2, a2, s);
          if (el == 0.0) continue;
          double r = 0.0;
          for (int u = 0; u < Sl; ++u) r += g[(size_t)s * S + u] * Eval(t, b, l + 2, q - 1, u, c2);
          sum += el * r;
        }
        return m.win[l1 + l2] * sum;
      });
      // hairpin interior enters the same way: XE += wh(d-1) E(p+1,q-1)
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
        double sum = 0.0;
        for (int s = 0; s < Sk; ++s)
          sum += Eval(t, b, p, k - 1, a1, s) * b.QBS[(size_t)(t.off[k] + s) * S + t.off[q + 1] + c1];
        return m.wbu[l1] * sum;
      }
      const int l2 = tt - 28, l = q - l2;  // right bulge
      if (l2 > maxint || l - p < mh1) return 0.0;
      const int Sl = t.sig[l + 1];
      double sum = 0.0;
      for (int u = 0; u < Sl; ++u)
        sum += b.QBS[(size_t)(t.off[p] + a1) * S + t.off[l + 1] + u] * Eval(t, b, l + 1, q, u, c1);
      return m.wbu[l2] * sum;
    });
    // ---- Z1: l1 = 1, l2 >= 2 ------------------------------------------------------------------------
    warp_terms(lane, nLp * Sq, 28, sc.Z1, [&](int e, int tt) {
      const int lst = e / Sq, c2 = e % Sq;
      const int l2 = tt + 2, l = q - l2;
      if (1 + l2 > maxint || l - (p + 1) < mh1) return 0.0;
      const int Sl = t.sig[l + 2];
      const double* dd = b.D1 + (size_t)(loffp + lst) * S + t.off[l + 2];
      double sum = 0.0;
      for (int u = 0; u < Sl; ++u) sum += dd[u] * Eval(t, b, l + 2, q - 1, u, c2);
      return m.win[1 + l2] * sum;
    });
    // ---- Z2: l2 = 1, l1 >= 2 ------------------------------------------------------------------------
    warp_terms(lane, Sp1 * nRq, 28, sc.Z2, [&](int e, int tt) {
      const int a2 = e / nRq, r = e % nRq;
      const int l1 = tt + 2, k = p + l1;
      if (l1 + 1 > maxint || (q - 1) - k < mh1) return 0.0;
      const int Sk = t.sig[k - 1];
      double sum = 0.0;
      for (int s = 0; s < Sk; ++s)
        sum += Eval(t, b, p + 1, k - 2, a2, s) * b.D2[(size_t)(t.off[k - 1] + s) * RS + roffq + r];
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

  // ---- M2(i,j) = sum_k Qm(i,k-1) Qm1(k,j): contiguous-row dot products; Qm = Qml + M2 --------------------
  {
    const int kb0 = t.off[i + 1], kb1 = offj1;
    double mx = 0.0;
    for (int e = 0; e < Si * Sj1; ++e) {
      const int a = e / Sj1, c = e % Sj1;
      const double* A = b.QM + (size_t)(offi + a) * S;
      const double* Bt = b.QM1T + (size_t)(offj1 + c) * S;
      double acc = 0.0;
      for (int kb = kb0 + lane; kb < kb1; kb += 32) acc += A[kb] * Bt[kb];
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      const double qm = sc.V1[e] + acc;
      if (lane == 0) {
        b.M2[(size_t)(offi + a) * S + offj1 + c] = acc;
        b.QM[(size_t)(offi + a) * S + offj1 + c] = qm;
      }
      mx = fmax(mx, qm);
    }
    if (lane == 0) b.cellexp[i] = mx > 0.0 ? ilogb(mx) : -100000;
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

__global__ void __launch_bounds__(CDZ_WARPS * 32) cell_kernel(const Ctx* ctxs, int d, int scr) {
  extern __shared__ double smem[];
  __shared__ CModel cm;
  const Ctx& cx = ctxs[blockIdx.y];
  {
    const int* src = (const int*)cx.cm;
    int* dst = (int*)&cm;
    for (int k = threadIdx.x; k < (int)(sizeof(CModel) / 4); k += blockDim.x) dst[k] = src[k];
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * CDZ_WARPS + warp;
  if (i + d >= cx.tt.n) return;
  Scratch sc = carve_scratch(smem + (size_t)warp * scr, cx.tt.MS, cm.nps, cx.tt.maxL, cx.tt.maxR);
  compute_cell(cx.tt, cx.tab, cm, sc, lane, i, i + d);
}

// Qext(j) = Qext(j-1) Tbar_j + sum_k Qext(k-1) Qbs(k,j); Z = sum_c Qext(n-1)[c]  (eq 3.7; App. A.3)
__global__ void __launch_bounds__(1024) exterior_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.x];
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const int n = t.n, S = t.S, MS = t.MS;
  const int mh1 = cx.cm->min_hairpin + 1;
  __shared__ double red[32][CDZ_MAX_BOND];
  // Qext is addressed by bond index: QX[off[k]+s] = Qext(k-1)[s]
  double* QX = b.Qext;
  if (threadIdx.x == 0) QX[0] = 1.0;
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int j = 0; j < n; ++j) {
    const int Sj1 = t.sig[j + 1];
    const int kend = j - mh1 >= 0 ? t.off[j - mh1 + 1] : 0;  // bonds of positions k <= j - mh1
    double acc[CDZ_MAX_BOND];
#pragma unroll
    for (int c = 0; c < CDZ_MAX_BOND; ++c) acc[c] = 0.0;
    for (int kb = threadIdx.x; kb < kend; kb += blockDim.x) {
      const double q = QX[kb];
      const double* row = b.QBS + (size_t)kb * S + t.off[j + 1];
#pragma unroll
      for (int c = 0; c < CDZ_MAX_BOND; ++c)
        if (c < Sj1) acc[c] += q * row[c];
    }
#pragma unroll
    for (int c = 0; c < CDZ_MAX_BOND; ++c) {
      for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
      if (lane == 0) red[warp][c] = acc[c];
    }
    __syncthreads();
    if (threadIdx.x < Sj1) {
      const int c = threadIdx.x;
      double v = 0.0;
      for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[w][c];
      const int Sj = t.sig[j];
      for (int s = 0; s < Sj; ++s) v += QX[t.off[j] + s] * t.Tbar[((size_t)j * MS + s) * MS + c];
      QX[t.off[j + 1] + c] = v;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double Z = 0.0;
    for (int c = 0; c < t.sig[n]; ++c) Z += QX[t.off[n] + c];
    const double ls = 0.6931471805599453 * (double)b.scale[n];
    b.result[0] = log(Z) + ls;
    b.result[1] = Z;
    b.result[2] = ls;
  }
}

__global__ void init_kernel(const Ctx* ctxs) {
  const Ctx& cx = ctxs[blockIdx.y];
  const int n = cx.tt.n;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k <= n + 1; k += gridDim.x * blockDim.x) {
    cx.tab.scale[k] = 0;
    if (k <= n) cx.tab.cellexp[k] = -100000;
    if (k < 64) cx.tab.ctrl[k] = 0;
  }
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
  // contexts of a batch must be contiguous on the device: stage them into the first handle's workspace? No:
  // each handle holds its own Ctx; for B > 1 we build a temporary array.
  int nmax = 0, MS = 1, maxL = 1, maxR = 1, nps = 6;
  for (int b = 0; b < B; ++b) {
    nmax = ts[b]->tt->n > nmax ? ts[b]->tt->n : nmax;
    MS = ts[b]->tt->MS > MS ? ts[b]->tt->MS : MS;
    maxL = ts[b]->tt->maxL > maxL ? ts[b]->tt->maxL : maxL;
    maxR = ts[b]->tt->maxR > maxR ? ts[b]->tt->maxR : maxR;
    if (ts[b]->model->c.nps > nps) nps = ts[b]->model->c.nps;
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
  const size_t smem = (size_t)scr * CDZ_WARPS * sizeof(double);
  CDZ_CUDA(cudaFuncSetAttribute(cell_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  init_kernel<<<dim3(8, B), 256, 0, st>>>(d_ctxs);
  for (int d = 0; d < nmax; ++d) {
    const int cells = nmax - d;
    dim3 grid((cells + CDZ_WARPS - 1) / CDZ_WARPS, B);
    cell_kernel<<<grid, CDZ_WARPS * 32, smem, st>>>(d_ctxs, d, scr);
  }
  exterior_kernel<<<B, 1024, 0, st>>>(d_ctxs);
  CDZ_CUDA(cudaGetLastError());
  if (tmp) CDZ_CUDA(cudaFreeAsync(tmp, st));
  return CDZ_OK;
}
