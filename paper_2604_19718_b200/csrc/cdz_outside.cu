// cdz_outside.cu -- outside (adjoint) pass over the stored inside tables: base-pair probabilities (sm_100a).
//
//   P(i.j) = sum_{a,x,y,c} Qb(i,j)[a,x,y,c] * dZ/dQb(i,j)[a,x,y,c] / Z            (eq 2.5 line 85; eq 4.1;
//                                                                                 SURVEY 8a-9 "outside / adjoint pass")
// The adjoint tables are gathered diagonal by diagonal, d = n-1 .. 0, from the cells that use cell (i,j) in the plain
// recursion of DESIGN.md section 3:
//   Qext-bar(k)   = Tbar_k Qext-bar(k+1) + sum_{j>=k} Qbs(k,j) Qext-bar(j+1),    Qext-bar(n) = 1/Z
//   Qm-bar(i,j)   = sum_{j'>j} M2-bar(i,j') Qm1(j+1,j')^T
//   M2-bar(i,j)   = Qm-bar(i,j) + w_a w_c sum_{x,y} I(i-1,j+1)[x,y]
//   Qml-bar(i,j)  = Qm-bar(i,j) + w_b Tbar_{i-1}^T Qml-bar(i-1,j)
//   Qm1-bar(i,j)  = Qml-bar(i,j) + w_b Qm1-bar(i,j+1) Tbar_{j+1}^T + sum_{i'<i} Qm(i',i-1)^T M2-bar(i',j)
//   Qbs-bar(i,j)  = w_c Qm1-bar(i,j) + Qext(i-1)^T Qext-bar(j+1)
//   Qb-bar(k,l)   = Qbs-bar(k,l) + sum over the closing pairs (i,j) = (k-1-l1, l+1+l2), l1+l2 <= 30, of the stack / bulge / interior
//                   term of Qb(i,j) differentiated with respect to Qb(k,l)
//   I(i,j)[x,y;a',c'] = sum_{a,c} T_i[a,x,a'] T_j[c',y,c] Qb-bar(i,j)[a,x,y,c]   (adjoint of `inner`),
//   G(i,j)[a',u,v,c'] = sum_{x,y} I(i,j)[x,y;a',c'] e^{-beta tmm[p(x,y)][u][v]}  (closing mismatch applied once per cell).
// All tables are the scaled ones the inside pass leaves behind: scaling every core by a power of two is a change of the
// operator weights under which the recursion is unchanged, and the probabilities are ratios.
// This version is a plain gather (one CTA per cell, one launch per diagonal, no tensor cores); the interior-loop term goes through
// per-closing-pair tables H / H1 / H2 (loop-side operators pre-contracted with G), so the inner cell only sums bond-indexed products.
#include "cdz_internal.h"

namespace {

constexpr int OT = 256;    // threads per CTA
constexpr int OPV = 1024;   // doubles of the per-operator scratch of the interior-loop term
constexpr int OZC = OPV / CDZ_MAX_BOND;  // operators per pass
constexpr int ORING = 34;  // diagonals of I / G / H / H1 / H2 kept: a closing pair lies at most 32 diagonals above its inner pair

struct Adj {
  double *AB, *AM2, *AML, *AM1, *AX, *IB, *G, *H, *H1, *H2;
};

// Qext-bar, sequential over bond positions k = n .. 0 (one CTA)
__global__ void __launch_bounds__(OT) oext_kernel(const Ctx* ctx, Adj A) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const int n = t.n, S = t.S, MS = t.MS;
  __shared__ double part[OT];
  __shared__ double zinv;
  if (threadIdx.x == 0) {
    double Z = 0.0;
    for (int c = 0; c < t.sig[n]; ++c) Z += b.Qext[t.off[n] + c];
    zinv = 1.0 / Z;
  }
  __syncthreads();
  if (threadIdx.x < MS) A.AX[(size_t)n * MS + threadIdx.x] = threadIdx.x < t.sig[n] ? zinv : 0.0;
  __syncthreads();
  const int grp = threadIdx.x / CDZ_MAX_BOND, s = threadIdx.x % CDZ_MAX_BOND, ngrp = OT / CDZ_MAX_BOND;
  for (int k = n - 1; k >= 0; --k) {
    double acc = 0.0;
    if (s < t.sig[k]) {
      for (int j = k + grp; j < n; j += ngrp) {
        const double* q = b.QBS + (size_t)(t.off[k] + s) * S + t.off[j + 1];
        const double* ax = A.AX + (size_t)(j + 1) * MS;
        for (int c = 0; c < t.sig[j + 1]; ++c) acc += q[c] * ax[c];
      }
    }
    part[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x < MS) {
      double v = 0.0;
      if (threadIdx.x < t.sig[k]) {
        for (int g = 0; g < ngrp; ++g) v += part[g * CDZ_MAX_BOND + threadIdx.x];
        for (int c = 0; c < t.sig[k + 1]; ++c)
          v += t.Tbar[((size_t)k * MS + threadIdx.x) * MS + c] * A.AX[(size_t)(k + 1) * MS + c];
      }
      A.AX[(size_t)k * MS + threadIdx.x] = v;
    }
    __syncthreads();
  }
}

struct OV {
  const DevTT& t;
  const DevTab& b;
  __device__ double E(int p, int q, int a, int c) const {
    if (q < p) return a == c ? 1.0 : 0.0;
    return b.EM[(size_t)(t.off[p] + a) * t.S + t.off[q + 1] + c];
  }
};

// deterministic block sum: every thread holds the partial of entry e = tid % nent, group tid / nent; returns the total to tid < nent
__device__ __forceinline__ double group_total(double* part, double v, int nent) {
  __syncthreads();
  part[threadIdx.x] = v;
  __syncthreads();
  double s = 0.0;
  if ((int)threadIdx.x < nent)
    for (int g = 0; g * nent + (int)threadIdx.x < OT; ++g)
      if (g < OT / nent) s += part[g * nent + threadIdx.x];
  return s;
}

// one diagonal d of the outside pass: CTA = cell (i, j = i + d)
__global__ void __launch_bounds__(OT) ocell_kernel(const Ctx* ctx, Adj A, int d, double* __restrict__ bpp) {
  const DevTT& t = ctx->tt;
  const DevTab& b = ctx->tab;
  const CModel& m = *ctx->cm;
  const OV V{t, b};
  const int n = t.n, S = t.S, RS = t.RS, MS = t.MS, MS2 = MS * MS, tid = threadIdx.x;
  const int i = blockIdx.x, j = i + d;
  const int Si = t.sig[i], Sj1 = t.sig[j + 1], offi = t.off[i], offj1 = t.off[j + 1];
  const int nent = Si * Sj1;
  __shared__ double part[OT];
  __shared__ double am[64], aml[64], abs_[64], ab[256], ibs[16 * 64];
  __shared__ uint8_t lp1[128], lp2[128];
  __shared__ double pv[OPV], pvg[64];
  __shared__ int nlp;
  if (tid == 0) {
    int c = 0;
    for (int l1 = 0; l1 <= m.max_interior; ++l1)
      for (int l2 = 0; l1 + l2 <= m.max_interior; ++l2)
        if (l1 == 0 || l2 == 0) { lp1[c] = (uint8_t)l1; lp2[c] = (uint8_t)l2; ++c; }  // stack + bulges; interior loops below
    nlp = c;
  }
  const int ngrp = OT / nent, e = tid % nent, grp = tid / nent;
  const bool act = grp < ngrp;
  const int ea = e / Sj1, ec = e % Sj1;
  // ---- Qm-bar(i,j)[a,s] = sum_{j'>j} sum_c M2-bar(i,j')[a,c] Qm1(j+1,j')[s,c]
  {
    double acc = 0.0;
    if (act)
      for (int jp = j + 1 + grp; jp < n; jp += ngrp) {
        const int o = t.off[jp + 1];
        const double* x = A.AM2 + (size_t)(offi + ea) * S + o;
        const double* q = b.QM1T + (size_t)o * S + offj1 + ec;
        for (int c = 0; c < t.sig[jp + 1]; ++c) acc += x[c] * q[(size_t)c * S];
      }
    const double v = group_total(part, acc, nent);
    if (tid < nent) am[tid] = v;
  }
  __syncthreads();
  if (tid < nent) {
    // ---- M2-bar = Qm-bar + w_a w_c sum_{x,y} I(i-1,j+1)[x,y]
    double v = am[tid];
    if (i >= 1 && j + 1 <= n - 1) {
      const double* ib = A.IB + ((size_t)((d + 2) % ORING) * n + (i - 1)) * 16 * MS2 + ea * MS + ec;
      double s = 0.0;
      for (int sl = 0; sl < m.nps; ++sl) s += ib[sl * MS2];
      v += m.wac * s;
    }
    A.AM2[(size_t)(offi + ea) * S + offj1 + ec] = v;
    // ---- Qml-bar = Qm-bar + w_b Tbar_{i-1}^T Qml-bar(i-1,j)
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
  // ---- Qm1-bar = Qml-bar + w_b Qm1-bar(i,j+1) Tbar_{j+1}^T + sum_{i'<i} Qm(i',i-1)^T M2-bar(i',j)
  {
    double acc = 0.0;
    if (act)
      for (int ip = grp; ip < i; ip += ngrp) {
        const int o = t.off[ip];
        for (int a2 = 0; a2 < t.sig[ip]; ++a2)
          acc += b.QM[(size_t)(o + a2) * S + offi + ea] * A.AM2[(size_t)(o + a2) * S + offj1 + ec];
      }
    const double v = group_total(part, acc, nent);
    if (tid < nent) {
      double w = aml[tid] + v;
      if (j + 1 <= n - 1) {
        double s = 0.0;
        for (int c2 = 0; c2 < t.sig[j + 2]; ++c2)
          s += A.AM1[(size_t)(offi + ea) * S + t.off[j + 2] + c2] * t.Tbar[((size_t)(j + 1) * MS + ec) * MS + c2];
        w += m.wb * s;
      }
      A.AM1[(size_t)(offi + ea) * S + offj1 + ec] = w;
      // ---- Qbs-bar = w_c Qm1-bar + Qext(i-1)^T Qext-bar(j+1)
      abs_[tid] = m.wc * w + b.Qext[offi + ea] * A.AX[(size_t)(j + 1) * MS + ec];
    }
  }
  __syncthreads();
  // ---- Qb-bar(k,l), (k,l) = this cell; closing pairs (i0,j0) = (k-1-l1, l+1+l2)
  const int k = i, l = j;
  const int nL = t.loff[k + 1] - t.loff[k], nR = t.roff[l + 1] - t.roff[l], npair = nL * nR;
  const bool closable = d >= m.min_hairpin + 1;
  // ---- interior loops l1, l2 >= 1 of the closing pairs (i0,j0) = (k-1-l1, l+1+l2).  With z2 at k-1 and z1' at l+1 the operators next to
  //      the inner pair,   Qb-bar(k,l)[s,x',y',t] += sum_{z2: c = s} sum_{z1': a = t} e^{-beta tmm[p(y',x')][b(z1')][b(z2)]} x_z2 x_z1' * in(z2,z1'),
  //      in = win[2] G(k-2,l+2)[a(z2),b(z2),b(z1'),c(z1')]  (1 x 1)  +  pv1[z2,c(z1')]  (l1 = 1)  +  pv2[z1',a(z2)]  (l2 = 1)  +  pvg[a(z2),c(z1')]
  //      where the loop-side operators of the closing pair were pre-contracted with G by the closing cell (H, H1, H2 below) and the
  //      unpaired stretches are E products.  Every sum runs in a fixed order: deterministic.
  double accI = 0.0;
  if (closable && k >= 2 && l + 2 <= n - 1) {
    const int e2 = tid % npair;
    const int ll = e2 / nR, rr = e2 % nR;
    const int s = t.ls_a[t.loff[k] + ll], xp = t.ls_x[t.loff[k] + ll];
    const int yp = t.rs_y[t.roff[l] + rr], tt_ = t.rs_c[t.roff[l] + rr];
    const bool mine = tid < npair && m.pslot[xp * 4 + yp] >= 0;
    const int Pin_il = m.ptype[yp * 4 + xp];
    const int z2b = t.opstart[k - 1], z1pb = t.opstart[l + 1], nz1p = t.opstart[l + 2] - z1pb;
    const int MI = m.max_interior;
    // l1, l2 >= 2: both side stretches are E products, so the term depends on (z2, z1') only through the bonds a(z2), c(z1'):
    //   pvg[a2,c1'] = sum_{l1,l2>=2} win[l1+l2] sum_{c1,a2'} E(i0+2,k-2)[c1,a2] H(i0,j0)[c1,a2'] E(l+2,j0-2)[c1',a2']
    const int Sk1 = t.sig[k - 1], Sl2 = t.sig[l + 2], nentg = Sk1 * Sl2;
    {
      const int eg = tid % nentg, gg = tid / nentg, ngg = OT / nentg;
      const int a2 = eg / Sl2, c1p = eg % Sl2;
      double acc = 0.0;
      if (gg < ngg)
        for (int l1 = 2 + gg; l1 <= MI - 2; l1 += ngg) {
          const int i0 = k - 1 - l1;
          if (i0 < 0) break;
          const int S1 = t.sig[i0 + 2];
          for (int l2 = 2; l1 + l2 <= MI; ++l2) {
            const int j0 = l + 1 + l2;
            if (j0 > n - 1) break;
            const int S2 = t.sig[j0 - 1];
            const double* H = A.H + ((size_t)((j0 - i0) % ORING) * n + i0) * MS2;
            double in = 0.0;
            for (int c1 = 0; c1 < S1; ++c1) {
              const double wl = V.E(i0 + 2, k - 2, c1, a2);
              if (wl == 0.0) continue;
              double r = 0.0;
              for (int a2p = 0; a2p < S2; ++a2p) r += H[c1 * MS + a2p] * V.E(l + 2, j0 - 2, c1p, a2p);
              in += wl * r;
            }
            acc += m.win[l1 + l2] * in;
          }
        }
      const double tot = group_total(part, acc, nentg);
      if (tid < nentg) pvg[tid] = tot;
    }
    __syncthreads();  // pvg
    // 1 x 1 loops (closing pair (k-2, l+2): G directly) and the generic part
    const int nz2 = t.opstart[k] - z2b;
    if (mine) {
      const double* G11 = A.G + ((size_t)(((l + 2) - (k - 2)) % ORING) * n + (k - 2)) * 16 * MS2;
      for (int z2 = z2b; z2 < z2b + nz2; ++z2) {
        if (t.op_c[z2] != s) continue;
        for (int z1p = z1pb; z1p < z1pb + nz1p; ++z1p) {
          if (t.op_a[z1p] != tt_) continue;
          accI += m.wtm[Pin_il][t.op_b[z1p]][t.op_b[z2]] * t.op_x[z2] * t.op_x[z1p] *
                  (pvg[t.op_a[z2] * Sl2 + t.op_c[z1p]] +
                   m.win[2] * G11[(t.op_b[z2] * 4 + t.op_b[z1p]) * MS2 + t.op_a[z2] * MS + t.op_c[z1p]]);
        }
      }
    }
    // l1 = 1, l2 >= 2: z1 = z2 carries both left mismatches; the right side is an E product ->
    //   pv[z2,c1'] = sum_{l2} win[1+l2] sum_{a2'} E(l+2,j0-2)[c1',a2'] H1(k-2,j0)[a(z2),b(z2),a2']
    for (int zb = 0; zb < nz2; zb += OZC) {
      const int zc = min(OZC, nz2 - zb);
      for (int e = tid; e < zc * Sl2; e += OT) {
        const int z2 = z2b + zb + e / Sl2, c1p = e % Sl2, i0 = k - 2;
        double v = 0.0;
        for (int l2 = 2; l2 <= MI - 1; ++l2) {
          const int j0 = l + 1 + l2;
          if (j0 > n - 1) break;
          const double* H1 = A.H1 + ((size_t)((j0 - i0) % ORING) * n + i0) * 4 * MS2 + (t.op_b[z2] * MS + t.op_a[z2]) * MS;
          const int S2 = t.sig[j0 - 1];
          double r = 0.0;
          for (int a2p = 0; a2p < S2; ++a2p) r += V.E(l + 2, j0 - 2, c1p, a2p) * H1[a2p];
          v += m.win[1 + l2] * r;
        }
        pv[e] = v;
      }
      __syncthreads();
      if (mine)
        for (int z2 = z2b + zb; z2 < z2b + zb + zc; ++z2) {
          if (t.op_c[z2] != s) continue;
          for (int z1p = z1pb; z1p < z1pb + nz1p; ++z1p) {
            if (t.op_a[z1p] != tt_) continue;
            accI += m.wtm[Pin_il][t.op_b[z1p]][t.op_b[z2]] * t.op_x[z2] * t.op_x[z1p] * pv[(z2 - z2b - zb) * Sl2 + t.op_c[z1p]];
          }
        }
      __syncthreads();
    }
    // l2 = 1, l1 >= 2: z2' = z1' carries both right mismatches ->
    //   pv[z1',a2] = sum_{l1} win[l1+1] sum_{c1} E(i0+2,k-2)[c1,a2] H2(i0,l+2)[c1,b(z1'),c(z1')]
    for (int zb = 0; zb < nz1p; zb += OZC) {
      const int zc = min(OZC, nz1p - zb);
      for (int e = tid; e < zc * Sk1; e += OT) {
        const int z1p = z1pb + zb + e / Sk1, a2 = e % Sk1, j0 = l + 2;
        double v = 0.0;
        for (int l1 = 2; l1 <= MI - 1; ++l1) {
          const int i0 = k - 1 - l1;
          if (i0 < 0) break;
          const double* H2 = A.H2 + ((size_t)((j0 - i0) % ORING) * n + i0) * 4 * MS2 + (t.op_b[z1p] * MS) * MS + t.op_c[z1p];
          const int S1 = t.sig[i0 + 2];
          double r = 0.0;
          for (int c1 = 0; c1 < S1; ++c1) r += V.E(i0 + 2, k - 2, c1, a2) * H2[c1 * MS];
          v += m.win[l1 + 1] * r;
        }
        pv[e] = v;
      }
      __syncthreads();
      if (mine)
        for (int z1p = z1pb + zb; z1p < z1pb + zb + zc; ++z1p) {
          if (t.op_a[z1p] != tt_) continue;
          for (int z2 = z2b; z2 < z2b + nz2; ++z2) {
            if (t.op_c[z2] != s) continue;
            accI += m.wtm[Pin_il][t.op_b[z1p]][t.op_b[z2]] * t.op_x[z2] * t.op_x[z1p] * pv[(z1p - z1pb - zb) * Sk1 + t.op_a[z2]];
          }
        }
      __syncthreads();
    }
  }
  {
    const int ng2 = OT / npair, e2 = tid % npair, g2 = tid / npair;
    const int ll = e2 / nR, rr = e2 % nR;
    const int s = t.ls_a[t.loff[k] + ll], xp = t.ls_x[t.loff[k] + ll];
    const int yp = t.rs_y[t.roff[l] + rr], tt_ = t.rs_c[t.roff[l] + rr];
    const bool pairable = m.pslot[xp * 4 + yp] >= 0;
    double acc = 0.0;
    if (g2 < ng2 && closable && pairable) {
      const int Pin_st = m.ptype[xp * 4 + yp];  // inner pair as (phi_k, phi_l): stacks and size-1 bulges
      for (int q = g2; q < nlp; q += ng2) {
        const int l1 = lp1[q], l2 = lp2[q];
        const int i0 = k - 1 - l1, j0 = l + 1 + l2;
        if (i0 < 0 || j0 > n - 1) continue;
        const int dd = j0 - i0;
        const int Sa = t.sig[i0 + 1], Sc = t.sig[j0];
        const double* ib = A.IB + ((size_t)(dd % ORING) * n + i0) * 16 * MS2;
        if (l1 == 0 && l2 == 0) {
          for (int sl = 0; sl < m.nps; ++sl)
            acc += m.wst[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][Pin_st] * ib[sl * MS2 + s * MS + tt_];
        } else if (l2 == 0) {
          // left bulge: sum_{a'} E(i0+1,k-1)[a',s] I[x,y;a',t]
          for (int sl = 0; sl < m.nps; ++sl) {
            const double w = m.wbu[l1] * (l1 == 1 ? m.wst[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][Pin_st] : 1.0);
            double v = 0.0;
            for (int a = 0; a < Sa; ++a) v += V.E(i0 + 1, k - 1, a, s) * ib[sl * MS2 + a * MS + tt_];
            acc += w * v;
          }
        } else if (l1 == 0) {
          // right bulge: sum_{c'} I[x,y;s,c'] E(l+1,j0-1)[t,c']
          for (int sl = 0; sl < m.nps; ++sl) {
            const double w = m.wbu[l2] * (l2 == 1 ? m.wst[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][Pin_st] : 1.0);
            double v = 0.0;
            for (int c = 0; c < Sc; ++c) v += ib[sl * MS2 + s * MS + c] * V.E(l + 1, j0 - 1, tt_, c);
            acc += w * v;
          }
        }
      }
    }
    const double v = group_total(part, acc, npair);
    if (tid < npair) {
      double w = 0.0;
      if (closable && pairable) w = v + accI + abs_[s * Sj1 + tt_];
      ab[tid] = w;
      A.AB[(size_t)(t.loff[k] + ll) * RS + t.roff[l] + rr] = w;
      part[tid] = w * b.QB[(size_t)(t.loff[k] + ll) * RS + t.roff[l] + rr];
    }
    __syncthreads();
    if (tid == 0) {
      double p = 0.0;
      for (int q = 0; q < npair; ++q) p += part[q];
      if (d > 0) bpp[(size_t)i * n + j] = p;
    }
  }
  __syncthreads();
  // ---- I(i,j)[slot][a'][c'] and G(i,j)[u,v][a'][c'] for the inner cells of this pair
  const int Sa = t.sig[i + 1], Sc = t.sig[j];
  double* ibo = A.IB + ((size_t)(d % ORING) * n + i) * 16 * MS2;
  double* go = A.G + ((size_t)(d % ORING) * n + i) * 16 * MS2;
  for (int q = tid; q < 16 * MS2; q += OT) {
    const int sl = q / MS2, ap = (q % MS2) / MS, cp = q % MS;
    double v = 0.0;
    if (sl < m.nps && ap < Sa && cp < Sc && closable && d >= 1) {
      const int x = m.slot_x[sl], y = m.slot_y[sl];
      for (int z = t.opstart[i]; z < t.opstart[i + 1]; ++z) {
        if (t.op_b[z] != x || t.op_c[z] != ap) continue;
        for (int zz = t.opstart[j]; zz < t.opstart[j + 1]; ++zz) {
          if (t.op_b[zz] != y || t.op_a[zz] != cp) continue;
          v += t.op_x[z] * t.op_x[zz] * ab[t.op_l[z] * nR + t.op_r[zz]];
        }
      }
    }
    ibs[q] = v;
    ibo[q] = v;
  }
  __syncthreads();
  for (int q = tid; q < 16 * MS2; q += OT) {
    const int uv = q / MS2, r = q % MS2;
    double v = 0.0;
    for (int sl = 0; sl < m.nps; ++sl)
      v += ibs[sl * MS2 + r] * m.wtm[m.ptype[m.slot_x[sl] * 4 + m.slot_y[sl]]][uv >> 2][uv & 3];
    go[q] = v;
  }
  // ---- H(i,j)[c1,a2'] = sum_{z1 at i+1: c = c1} sum_{z2' at j-1: a = a2'} x_z1 x_z2' G(i,j)[a(z1),b(z1),b(z2'),c(z2')]
  //      (both loop-side operators of an interior loop with l1, l2 >= 2 closed by this pair)
  __syncthreads();
  double* ho = A.H + ((size_t)(d % ORING) * n + i) * MS2;
  for (int q = tid; q < MS2; q += OT) {
    const int c1 = q / MS, a2p = q % MS;
    double v = 0.0;
    if (closable && j - 1 > i + 1)
      for (int z1 = t.opstart[i + 1]; z1 < t.opstart[i + 2]; ++z1) {
        if (t.op_c[z1] != c1) continue;
        const double* Gz = go + (t.op_b[z1] * 4) * MS2 + t.op_a[z1] * MS;
        for (int z2p = t.opstart[j - 1]; z2p < t.opstart[j]; ++z2p)
          if (t.op_a[z2p] == a2p) v += t.op_x[z1] * t.op_x[z2p] * Gz[t.op_b[z2p] * MS2 + t.op_c[z2p]];
      }
    ho[q] = v;
  }
  // ---- H1(i,j)[u,a,a2'] = sum_{z2' at j-1: a = a2'} x_z2' G[a,u,b(z2'),c(z2')]   (l1 = 1: the operator at i+1 stays open)
  //      H2(i,j)[v,c1,c'] = sum_{z1 at i+1: c = c1} x_z1 G[a(z1),b(z1),v,c']       (l2 = 1: the operator at j-1 stays open)
  double* h1o = A.H1 + ((size_t)(d % ORING) * n + i) * 4 * MS2;
  double* h2o = A.H2 + ((size_t)(d % ORING) * n + i) * 4 * MS2;
  for (int q = tid; q < 8 * MS2; q += OT) {
    const int which = q / (4 * MS2), r = q % (4 * MS2);
    const int uv = r / MS2, x1 = (r % MS2) / MS, x2 = r % MS;
    double v = 0.0;
    if (closable && j - 1 > i + 1) {
      if (which == 0) {  // u = uv, a = x1, a2' = x2
        for (int z2p = t.opstart[j - 1]; z2p < t.opstart[j]; ++z2p)
          if (t.op_a[z2p] == x2) v += t.op_x[z2p] * go[(uv * 4 + t.op_b[z2p]) * MS2 + x1 * MS + t.op_c[z2p]];
      } else {  // v = uv, c1 = x1, c' = x2
        for (int z1 = t.opstart[i + 1]; z1 < t.opstart[i + 2]; ++z1)
          if (t.op_c[z1] == x1) v += t.op_x[z1] * go[(t.op_b[z1] * 4 + uv) * MS2 + t.op_a[z1] * MS + x2];
      }
    }
    (which == 0 ? h1o : h2o)[r] = v;
  }
}

__global__ void unpaired_kernel(int n, double* __restrict__ bpp) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double s = 0.0;
  for (int j = i + 1; j < n; ++j) s += bpp[(size_t)i * n + j];
  for (int j = 0; j < i; ++j) s += bpp[(size_t)j * n + i];
  bpp[(size_t)i * n + i] = 1.0 - s;
}

}  // namespace

// Base-pair probabilities of a finished inside pass: bpp_dev [n][n], upper triangle P(i.j), diagonal P(i unpaired), lower triangle 0.
// Workspace (3 S x S + LS x RS adjoint tables, 34 diagonals of I / G / H / H1 / H2) is allocated for the call and freed before it returns.
int cdz_launch_outside(cdz_tables* t, double* bpp_dev, cudaStream_t st) {
  const cdz_tt* tt = t->tt;
  const size_t n = tt->n, S = tt->S, LS = tt->LS, RS = tt->RS, MS = tt->MS;
  const size_t nSS = S * S, nAB = LS * RS, nAX = (n + 1) * MS, nR = (size_t)ORING * n * 16 * MS * MS;
  const size_t nH = (size_t)ORING * n * MS * MS;
  const size_t total = 3 * nSS + nAB + nAX + 2 * nR + 9 * nH;
  double* ws = nullptr;
  if (cudaMalloc(&ws, total * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    cdz_set_error("cdz_marginals: out of device memory for the adjoint tables");
    return CDZ_ENOMEM;
  }
  Adj A;
  double* p = ws;
  A.AM2 = p; p += nSS;
  A.AML = p; p += nSS;
  A.AM1 = p; p += nSS;
  A.AB = p; p += nAB;
  A.AX = p; p += nAX;
  A.IB = p; p += nR;
  A.G = p; p += nR;
  A.H = p; p += nH;
  A.H1 = p; p += 4 * nH;
  A.H2 = p; p += 4 * nH;
  cudaError_t e = cudaMemsetAsync(ws, 0, total * sizeof(double), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(bpp_dev, 0, n * n * sizeof(double), st);
  if (e == cudaSuccess) {
    oext_kernel<<<1, OT, 0, st>>>(t->d_ctx, A);
    for (int d = (int)n - 1; d >= 0; --d) ocell_kernel<<<(unsigned)(n - d), OT, 0, st>>>(t->d_ctx, A, d, bpp_dev);
    unpaired_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>((int)n, bpp_dev);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(ws);
  if (e != cudaSuccess) {
    cdz_set_error(std::string("cdz_marginals (outside pass): ") + cudaGetErrorString(e));
    return CDZ_ECUDA;
  }
  return CDZ_OK;
}
