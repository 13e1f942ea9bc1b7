// cdz_sample.cu -- batched stochastic traceback (sm_100a): one warp per sample walks the stored inside tables
// and emits an exact sample (phi, s) ~ W(phi) exp(-E/kT) / Z  (PAPER.md S4c, Alg S4.4).
//
// Every decision lists its alternatives in the canonical order of DESIGN.md "Traceback order" and takes the
// first one whose running sum exceeds u * total, where u = U(seed, sample, kind, i, j) is a counter-based
// uniform.  Lanes evaluate 32 alternatives at a time (shuffle prefix scan), cheapest / likeliest segments first,
// and stop at the first hit, so the expensive interior-loop alternatives are only evaluated when needed.
#include <math.h>
#include <stdio.h>

#include <mutex>

#include "cdz_internal.h"

namespace {

enum { K_TOP = 0, K_EXT = 1, K_QB = 2, K_QM = 3, K_QML = 4, K_QM1 = 5, K_CHAIN = 6, K_HAIRPIN = 7, K_ILOOP = 8 };
enum { IT_QB = 0, IT_QM = 1, IT_QML = 2, IT_QM1 = 3 };

struct Item { int type, i, j; short a, x, y, c; };

__device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double uniform(uint64_t seed, uint64_t sample, uint64_t kind, uint64_t i, uint64_t j) {
  uint64_t h = seed;
  h = mix64(h + 0x9E3779B97F4A7C15ULL * (sample + 1));
  h = mix64(h + 0x9E3779B97F4A7C15ULL * (kind + 1));
  h = mix64(h + 0x9E3779B97F4A7C15ULL * (i + 1));
  h = mix64(h + 0x9E3779B97F4A7C15ULL * (j + 1));
  return (double)(h >> 11) * (1.0 / 9007199254740992.0);
}

struct Pick {
  double thr, run;
  int last;   // last positive alternative seen (global id), -1 if none
  int hit;    // chosen global id or -1
};

// scan `count` alternatives (ids base..base+count) of one segment; returns true when the pick is decided
template <typename F>
__device__ __forceinline__ bool scan_segment(int lane, Pick& pk, int base, int count, F weight) {
  for (int b0 = 0; b0 < count; b0 += 32) {
    const int idx = b0 + lane;
    double w = idx < count ? weight(idx) : 0.0;
    if (!(w > 0.0)) w = 0.0;
    double s = w;
    for (int o = 1; o < 32; o <<= 1) {
      double v = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += v;
    }
    const double cum = pk.run + s;
    const unsigned pos = __ballot_sync(0xffffffffu, w > 0.0);
    const unsigned hit = __ballot_sync(0xffffffffu, w > 0.0 && cum > pk.thr);
    if (pos) pk.last = base + b0 + 31 - __clz(pos);
    if (hit) { pk.hit = base + b0 + __ffs(hit) - 1; return true; }
    pk.run += __shfl_sync(0xffffffffu, s, 31);
  }
  return false;
}

template <typename F>
__device__ __forceinline__ double warp_total(int lane, int count, F weight) {
  double s = 0.0;
  for (int idx = lane; idx < count; idx += 32) { double w = weight(idx); if (w > 0.0) s += w; }
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  return s;
}

struct View {
  const DevTT& t;
  const DevTab& b;
  const CModel& m;
  __device__ double E(int p, int q, int a, int c) const {
    if (q < p) return a == c ? 1.0 : 0.0;
    return b.EM[(size_t)(t.off[p] + a) * t.S + t.off[q + 1] + c];
  }
  __device__ double QB(int i, int j, int a, int x, int y, int c) const {  // dense view of the state-list cell
    const int ll = t.lsidx[((size_t)i * t.MS + a) * 4 + x], rr = t.rsidx[((size_t)j * 4 + y) * t.MS + c];
    if (ll < 0 || rr < 0) return 0.0;
    const int l = t.loff[i] + ll, r = t.roff[j] + rr;
    if (l < 0 || r < 0) return 0.0;
    return b.QB[(size_t)l * t.RS + r];
  }
  __device__ bool can(int x, int y) const { return m.pslot[x * 4 + y] >= 0; }
  __device__ int pt(int x, int y) const { return m.ptype[x * 4 + y]; }
};

// weight of one sub-alternative of the loop closed by (i,j) with inner pair (k,l):
// left side index la, right side index ra (rectangular operator ranges), inner nucleotides (xp,yp).
// Outputs the bonds (s,t) of the inner cell and the operators chosen.
struct SideL { int z1, z2, u, up, s; double w; };
__device__ __forceinline__ SideL left_side(const View& V, int i, int k, int ap, int la) {
  const DevTT& t = V.t;
  const int l1 = k - i - 1;
  SideL r; r.z1 = r.z2 = -1; r.u = r.up = 0; r.s = ap; r.w = 1.0;
  if (l1 == 0) return r;
  if (l1 == 1) {
    const int z = t.opstart[i + 1] + la;
    r.z1 = z; r.u = r.up = t.op_b[z]; r.s = t.op_c[z];
    r.w = t.op_a[z] == ap ? t.op_x[z] : 0.0;
    return r;
  }
  const int n2 = t.opstart[k] - t.opstart[k - 1];
  const int z = t.opstart[i + 1] + la / n2, z2 = t.opstart[k - 1] + la % n2;
  r.z1 = z; r.z2 = z2; r.u = t.op_b[z]; r.up = t.op_b[z2]; r.s = t.op_c[z2];
  r.w = t.op_a[z] == ap ? t.op_x[z] * V.E(i + 2, k - 2, t.op_c[z], t.op_a[z2]) * t.op_x[z2] : 0.0;
  return r;
}
__device__ __forceinline__ int left_count(const DevTT& t, int i, int k) {
  const int l1 = k - i - 1;
  if (l1 == 0) return 1;
  const int n1 = t.opstart[i + 2] - t.opstart[i + 1];
  if (l1 == 1) return n1;
  return n1 * (t.opstart[k] - t.opstart[k - 1]);
}
// right side: z1 = operator at l+1 (v'), z2 = operator at j-1 (v); .u = v, .up = v', .s = t
__device__ __forceinline__ SideL right_side(const View& V, int j, int l, int cp, int ra) {
  const DevTT& t = V.t;
  const int l2 = j - l - 1;
  SideL r; r.z1 = r.z2 = -1; r.u = r.up = 0; r.s = cp; r.w = 1.0;
  if (l2 == 0) return r;
  if (l2 == 1) {
    const int z = t.opstart[j - 1] + ra;
    r.z1 = z; r.u = r.up = t.op_b[z]; r.s = t.op_a[z];
    r.w = t.op_c[z] == cp ? t.op_x[z] : 0.0;
    return r;
  }
  const int n2 = t.opstart[j] - t.opstart[j - 1];
  const int z = t.opstart[l + 1] + ra / n2, z2 = t.opstart[j - 1] + ra % n2;
  r.z1 = z; r.z2 = z2; r.u = t.op_b[z2]; r.up = t.op_b[z]; r.s = t.op_a[z];
  r.w = t.op_c[z2] == cp ? t.op_x[z] * V.E(l + 2, j - 2, t.op_c[z], t.op_a[z2]) * t.op_x[z2] : 0.0;
  return r;
}
__device__ __forceinline__ int right_count(const DevTT& t, int j, int l) {
  const int l2 = j - l - 1;
  if (l2 == 0) return 1;
  const int n2 = t.opstart[j] - t.opstart[j - 1];
  if (l2 == 1) return n2;
  return (t.opstart[l + 2] - t.opstart[l + 1]) * n2;
}
__device__ __forceinline__ double loop_factor(const View& V, int P, int l1, int l2, int xp, int yp, const SideL& L,
                                              const SideL& R) {
  const CModel& m = V.m;
  if (l1 == 0 && l2 == 0) return m.wst[P][V.pt(xp, yp)];
  if (l1 == 0 || l2 == 0) return m.wbu[l1 + l2] * (l1 + l2 == 1 ? m.wst[P][V.pt(xp, yp)] : 1.0);
  return m.win[l1 + l2] * m.wtm[P][L.u][R.u] * m.wtm[V.pt(yp, xp)][R.up][L.up];
}
// total weight of inner pair (k,l) for closing (i,j,x,y) with a' = ap, c' = cp (sequential, one lane).
// Same quantity as the explicit sum over side operators and inner nucleotides (the oracle's level A), evaluated from the
// pre-contracted tables the inside pass keeps: Qbs for bulges >= 2, the
// mismatch-dressed extensions DD / D1 / D2T / GI of Qb(k,l) for interior loops.
__device__ double iloop_total(const View& V, int i, int j, int k, int l, int P, int ap, int cp) {
  const DevTT& t = V.t;
  const DevTab& b = V.b;
  const CModel& m = V.m;
  const int l1 = k - i - 1, l2 = j - l - 1, MS = t.MS;
  const size_t S = (size_t)t.S, RS = (size_t)t.RS;
  if (l1 == 0 && l2 == 0) {
    double tot = 0.0;
    for (int sl = 0; sl < m.nps; ++sl) {
      const int xp = m.slot_x[sl], yp = m.slot_y[sl];
      tot += m.wst[P][V.pt(xp, yp)] * V.QB(k, l, ap, xp, yp, cp);
    }
    return tot;
  }
  if (l2 == 0 || l1 == 0) {
    const int len = l1 + l2;
    if (len >= 2) {
      double tot = 0.0;
      if (l2 == 0) {
        for (int s = 0; s < t.sig[k]; ++s) tot += V.E(i + 1, k - 1, ap, s) * b.QBS[(size_t)(t.off[k] + s) * S + t.off[l + 1] + cp];
      } else {
        for (int u = 0; u < t.sig[l + 1]; ++u) tot += b.QBS[(size_t)(t.off[k] + ap) * S + t.off[l + 1] + u] * V.E(l + 1, j - 1, u, cp);
      }
      return m.wbu[len] * tot;
    }
    // size-1 bulge: the stack term keeps the identity of the inner pair
    double tot = 0.0;
    for (int sl = 0; sl < m.nps; ++sl) {
      const int xp = m.slot_x[sl], yp = m.slot_y[sl];
      double q = 0.0;
      if (l2 == 0) {
        for (int s = 0; s < t.sig[k]; ++s) q += t.Tbar[((size_t)(i + 1) * MS + ap) * MS + s] * V.QB(k, l, s, xp, yp, cp);
      } else {
        for (int u = 0; u < t.sig[l + 1]; ++u) q += V.QB(k, l, ap, xp, yp, u) * t.Tbar[((size_t)(j - 1) * MS + u) * MS + cp];
      }
      tot += m.wst[P][V.pt(xp, yp)] * q;
    }
    return m.wbu[1] * tot;
  }
  // interior loops: mismatch at the closing pair from the operators at i+1 / j-1, the inner pair's mismatch is in the tables
  const int pl = k - 1, pr = l + 1;  // positions dressed onto Qb(k,l)
  double tot = 0.0;
  if (l1 == 1 && l2 == 1) {
    for (int lst = t.loff[pl]; lst < t.loff[pl + 1]; ++lst) {
      if (t.ls_a[lst] != ap) continue;
      for (int r = t.roff[pr]; r < t.roff[pr + 1]; ++r)
        if (t.rs_c[r] == cp) tot += m.wtm[P][t.ls_x[lst]][t.rs_y[r]] * b.DD[(size_t)lst * RS + r];
    }
  } else if (l1 == 1) {
    for (int lst = t.loff[pl]; lst < t.loff[pl + 1]; ++lst) {
      if (t.ls_a[lst] != ap) continue;
      const double* d1 = b.D1 + (size_t)lst * S + t.off[l + 2];
      for (int w = t.opstart[j - 1]; w < t.opstart[j]; ++w) {
        if (t.op_c[w] != cp) continue;
        double s = 0.0;
        for (int t2 = 0; t2 < t.sig[l + 2]; ++t2) s += d1[t2] * V.E(l + 2, j - 2, t2, t.op_a[w]);
        tot += t.op_x[w] * m.wtm[P][t.ls_x[lst]][t.op_b[w]] * s;
      }
    }
  } else if (l2 == 1) {
    for (int r = t.roff[pr]; r < t.roff[pr + 1]; ++r) {
      if (t.rs_c[r] != cp) continue;
      const double* d2 = b.D2T + (size_t)r * S + t.off[k - 1];
      for (int z = t.opstart[i + 1]; z < t.opstart[i + 2]; ++z) {
        if (t.op_a[z] != ap) continue;
        double s = 0.0;
        for (int s2 = 0; s2 < t.sig[k - 1]; ++s2) s += V.E(i + 2, k - 2, t.op_c[z], s2) * d2[s2];
        tot += t.op_x[z] * m.wtm[P][t.op_b[z]][t.rs_y[r]] * s;
      }
    }
  } else {
    const double* gi = b.GI + (size_t)t.off[k - 1] * S + t.off[l + 2];
    const int Sk = t.sig[k - 1], Sl = t.sig[l + 2];
    for (int z = t.opstart[i + 1]; z < t.opstart[i + 2]; ++z) {
      if (t.op_a[z] != ap) continue;
      for (int w = t.opstart[j - 1]; w < t.opstart[j]; ++w) {
        if (t.op_c[w] != cp) continue;
        double s = 0.0;
        for (int s2 = 0; s2 < Sk; ++s2) {
          const double el = V.E(i + 2, k - 2, t.op_c[z], s2);
          if (el == 0.0) continue;
          double r2 = 0.0;
          for (int t2 = 0; t2 < Sl; ++t2) r2 += gi[(size_t)s2 * S + t2] * V.E(l + 2, j - 2, t2, t.op_a[w]);
          s += el * r2;
        }
        tot += t.op_x[z] * t.op_x[w] * m.wtm[P][t.op_b[z]][t.op_b[w]] * s;
      }
    }
  }
  return m.win[l1 + l2] * tot;
}

__global__ void __launch_bounds__(128) sample_kernel(const Ctx* ctxp, int J, uint64_t seed, uint8_t* seq_out,
                                                     int32_t* pair_out, Item* stacks, int stack_cap) {
  __shared__ CModel cm;
  // per warp: the operators compatible with the boundary state of the element being decomposed (weights and inner bonds), see QB / ILOOP
  constexpr int CCAP = 40;
  __shared__ double s_cw[4][2][CCAP];
  __shared__ short s_cb[4][2][CCAP], s_cz[4][2][CCAP];
  const Ctx& cx = *ctxp;
  {
    const int* src = (const int*)cx.cm;
    int* dst = (int*)&cm;
    for (int k = threadIdx.x; k < (int)(sizeof(CModel) / 4); k += blockDim.x) dst[k] = src[k];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int smp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (smp >= J) return;
  const DevTT& t = cx.tt;
  const DevTab& b = cx.tab;
  const View V{t, b, cm};
  const int n = t.n, S = t.S, RS = t.RS;
  const int mh1 = cm.min_hairpin + 1, maxint = cm.max_interior;
  uint8_t* seq = seq_out + (size_t)smp * n;
  int32_t* pair = pair_out + (size_t)smp * n;
  Item* stk = stacks + (size_t)smp * stack_cap;
  int sp = 0;
  for (int k = lane; k < n; k += 32) { seq[k] = 255; pair[k] = -1; }
  __syncwarp();
  const double* QX = b.Qext;

  // ---- CHAIN(p,q,s,tend): unpaired stretch with fixed end bonds -------------------------------------
  auto chain = [&](int p, int q, int s, int tend) {
    int cur = s;
    for (int mp = p; mp <= q; ++mp) {
      const int z0 = t.opstart[mp], cnt = t.opstart[mp + 1] - z0;
      auto wf = [&](int k) {
        const int z = z0 + k;
        return t.op_a[z] == cur ? t.op_x[z] * V.E(mp + 1, q, t.op_c[z], tend) : 0.0;
      };
      Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
      pk.thr = uniform(seed, smp, K_CHAIN, mp, 0) * warp_total(lane, cnt, wf);
      scan_segment(lane, pk, 0, cnt, wf);
      const int z = z0 + (pk.hit >= 0 ? pk.hit : pk.last);
      if (lane == 0) seq[mp] = t.op_b[z];
      cur = t.op_c[z];
    }
  };

  // ---- TOP / EXT -------------------------------------------------------------------------------------
  int cb;
  {
    const int cnt = t.sig[n];
    auto wf = [&](int c) { return QX[t.off[n] + c]; };
    Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
    pk.thr = uniform(seed, smp, K_TOP, 0, 0) * warp_total(lane, cnt, wf);
    scan_segment(lane, pk, 0, cnt, wf);
    cb = pk.hit >= 0 ? pk.hit : pk.last;
  }
  int j = n - 1;
  while (j >= 0) {
    const int z0 = t.opstart[j], nops = t.opstart[j + 1] - z0;
    Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
    pk.thr = uniform(seed, smp, K_EXT, j, 0) * QX[t.off[j + 1] + cb];
    bool done = scan_segment(lane, pk, 0, nops, [&](int k) {
      const int z = z0 + k;
      return t.op_c[z] == cb ? QX[t.off[j] + t.op_a[z]] * t.op_x[z] : 0.0;
    });
    // pairs (k,j): alternatives over (left state of k) x (right states of j with c = cb), k ascending
    int nrc = 0;
    for (int r = t.roff[j]; r < t.roff[j + 1]; ++r) nrc += (t.rs_c[r] == cb);
    const int nls = j - mh1 >= 0 ? t.loff[j - mh1 + 1] : 0;  // left states of positions k <= j - mh1
    const int base = nops;
    auto pw = [&](int idx) {
      const int l = idx / nrc;
      int rr = idx % nrc, r = t.roff[j];
      for (;; ++r) if (t.rs_c[r] == cb) { if (rr == 0) break; --rr; }
      const int k = t.lspos[l];
      if (!V.can(t.ls_x[l], t.rs_y[r])) return 0.0;
      return QX[t.off[k] + t.ls_a[l]] * b.QB[(size_t)l * RS + r];
    };
    if (!done && nrc > 0) done = scan_segment(lane, pk, base, nls * nrc, pw);
    const int pick = pk.hit >= 0 ? pk.hit : pk.last;
    if (pick < nops) {
      const int z = z0 + pick;
      if (lane == 0) seq[j] = t.op_b[z];
      cb = t.op_a[z];
      j -= 1;
    } else {
      const int idx = pick - base;
      const int l = idx / nrc;
      int rr = idx % nrc, r = t.roff[j];
      for (;; ++r) if (t.rs_c[r] == cb) { if (rr == 0) break; --rr; }
      const int k = t.lspos[l];
      if (lane == 0) stk[sp] = Item{IT_QB, k, j, (short)t.ls_a[l], (short)t.ls_x[l], (short)t.rs_y[r], (short)cb};
      ++sp;
      cb = t.ls_a[l];
      j = k - 1;
    }
  }
  __syncwarp();

  while (sp > 0) {
    --sp;
    const Item it = stk[sp];
    __syncwarp();
    const int i = it.i;
    j = it.j;
    const int offi = t.off[i], offj1 = t.off[j + 1];
    if (it.type == IT_QM) {
      // {Qml(i,j)[a,c]}, then {k asc, s asc: Qm(i,k-1)[a,s] Qm1(k,j)[s,c]}
      Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
      pk.thr = uniform(seed, smp, K_QM, i, j) * b.QM[(size_t)(offi + it.a) * S + offj1 + it.c];
      bool done = scan_segment(lane, pk, 0, 1, [&](int) { return b.QML[(size_t)(offi + it.a) * S + offj1 + it.c]; });
      const int kb0 = t.off[i + 1];
      const double* A = b.QM + (size_t)(offi + it.a) * S;
      const double* Bt = b.QM1T + (size_t)(offj1 + it.c) * S;
      if (!done) scan_segment(lane, pk, 1, offj1 - kb0, [&](int k) { return A[kb0 + k] * Bt[kb0 + k]; });
      const int pick = pk.hit >= 0 ? pk.hit : pk.last;
      if (pick == 0) {
        if (lane == 0) stk[sp] = Item{IT_QML, i, j, it.a, 0, 0, it.c};
        ++sp;
      } else {
        const int kb = kb0 + pick - 1;
        const int k = t.bondpos[kb], s = kb - t.off[k];
        if (lane == 0) {
          stk[sp] = Item{IT_QM, i, k - 1, it.a, 0, 0, (short)s};
          stk[sp + 1] = Item{IT_QM1, k, j, (short)s, 0, 0, it.c};
        }
        sp += 2;
      }
    } else if (it.type == IT_QML) {
      // {Qm1(i,j)[a,c]}, then {z at i with a(z)=a: w_b x(z) Qml(i+1,j)[c(z),c]}
      const int z0 = t.opstart[i], nops = t.opstart[i + 1] - z0;
      Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
      pk.thr = uniform(seed, smp, K_QML, i, j) * b.QML[(size_t)(offi + it.a) * S + offj1 + it.c];
      scan_segment(lane, pk, 0, 1 + nops, [&](int k) {
        if (k == 0) return b.QM1T[(size_t)(offj1 + it.c) * S + offi + it.a];
        const int z = z0 + k - 1;
        if (t.op_a[z] != it.a || i + 1 > j) return 0.0;
        return cm.wb * t.op_x[z] * b.QML[(size_t)(t.off[i + 1] + t.op_c[z]) * S + offj1 + it.c];
      });
      const int pick = pk.hit >= 0 ? pk.hit : pk.last;
      if (pick == 0) {
        if (lane == 0) stk[sp] = Item{IT_QM1, i, j, it.a, 0, 0, it.c};
      } else {
        const int z = z0 + pick - 1;
        if (lane == 0) { seq[i] = t.op_b[z]; stk[sp] = Item{IT_QML, i + 1, j, (short)t.op_c[z], 0, 0, it.c}; }
      }
      ++sp;
    } else if (it.type == IT_QM1) {
      // {(x,y) lexicographic: w_c Qb(i,j)[a,x,y,c]}, then {z at j with c(z)=c: w_b Qm1(i,j-1)[a,a(z)] x(z)}
      const int z0 = t.opstart[j], nops = t.opstart[j + 1] - z0;
      Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
      pk.thr = uniform(seed, smp, K_QM1, i, j) * b.QM1T[(size_t)(offj1 + it.c) * S + offi + it.a];
      scan_segment(lane, pk, 0, 16 + nops, [&](int k) {
        if (k < 16) return V.can(k >> 2, k & 3) ? cm.wc * V.QB(i, j, it.a, k >> 2, k & 3, it.c) : 0.0;
        const int z = z0 + k - 16;
        if (t.op_c[z] != it.c || j - 1 < i) return 0.0;
        return cm.wb * b.QM1T[(size_t)(t.off[j] + t.op_a[z]) * S + offi + it.a] * t.op_x[z];
      });
      const int pick = pk.hit >= 0 ? pk.hit : pk.last;
      if (pick < 16) {
        if (lane == 0) stk[sp] = Item{IT_QB, i, j, it.a, (short)(pick >> 2), (short)(pick & 3), it.c};
      } else {
        const int z = z0 + pick - 16;
        if (lane == 0) { seq[j] = t.op_b[z]; stk[sp] = Item{IT_QM1, i, j - 1, it.a, 0, 0, (short)t.op_a[z]}; }
      }
      ++sp;
    } else {
      // ---- QB(i,j,a,x,y,c) -----------------------------------------------------------------------------
      const int x = it.x, y = it.y, d = j - i, P = V.pt(x, y);
      if (lane == 0) { seq[i] = (uint8_t)x; seq[j] = (uint8_t)y; pair[i] = j; pair[j] = i; }
      const int zi0 = t.opstart[i], ni = t.opstart[i + 1] - zi0, zj0 = t.opstart[j], nj = t.opstart[j + 1] - zj0;
      // The (z_i, z_j) alternatives with non-zero weight are the product of the operators at i with (a, b) = (it.a, x) and those at j with
      // (b, c) = (y, it.c), in list order.  Zero-weight alternatives never decide a pick, so only that product is
      // scanned: the two compatible lists are compacted once per decision (weight and inner bond of every entry) into shared memory.
      const int wrp = threadIdx.x >> 5;
      double* cwi = s_cw[wrp][0];
      double* cwj = s_cw[wrp][1];
      short* cai = s_cb[wrp][0];
      short* ccj = s_cb[wrp][1];
      int ci = 0, cj = 0;
      __syncwarp();
      for (int b0 = 0; b0 < ni; b0 += 32) {
        const int z = zi0 + b0 + lane;
        const bool ok = b0 + lane < ni && t.op_a[z] == it.a && t.op_b[z] == x;
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        const int pos = ci + __popc(m & ((1u << lane) - 1u));
        if (ok && pos < CCAP) { cwi[pos] = t.op_x[z]; cai[pos] = (short)t.op_c[z]; }
        ci += __popc(m);
      }
      for (int b0 = 0; b0 < nj; b0 += 32) {
        const int z = zj0 + b0 + lane;
        const bool ok = b0 + lane < nj && t.op_b[z] == y && t.op_c[z] == it.c;
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        const int pos = cj + __popc(m & ((1u << lane) - 1u));
        if (ok && pos < CCAP) { cwj[pos] = t.op_x[z]; ccj[pos] = (short)t.op_a[z]; }
        cj += __popc(m);
      }
      __syncwarp();
      const bool compact = ci <= CCAP && cj <= CCAP;  // (otherwise the rectangular space below; mismatching operators weigh 0)
      const int npair = compact ? ci * cj : ni * nj;
      auto zw = [&](int pz, int& ap, int& cp) {
        if (compact) {
          const int ki = pz / cj, kj = pz - ki * cj;
          ap = cai[ki]; cp = ccj[kj];
          return cwi[ki] * cwj[kj];
        }
        const int zi = zi0 + pz / nj, zj = zj0 + pz % nj;
        ap = t.op_c[zi]; cp = t.op_a[zj];
        if (t.op_a[zi] != it.a || t.op_b[zi] != x || t.op_b[zj] != y || t.op_c[zj] != it.c) return 0.0;
        return t.op_x[zi] * t.op_x[zj];
      };
      Pick pk; pk.run = 0.0; pk.last = -1; pk.hit = -1;
      pk.thr = uniform(seed, smp, K_QB, i, j) * V.QB(i, j, it.a, x, y, it.c);
      const int p = i + 1, q = j - 1;
      // segment 0: hairpin, per (z_i,z_j)
      const double wh = t.wh[d - 1];
      bool done = scan_segment(lane, pk, 0, npair, [&](int pz) {
        int ap, cp;
        const double w0 = zw(pz, ap, cp);
        if (w0 == 0.0) return 0.0;
        double s = 0.0;
        for (int zp = t.opstart[p]; zp < t.opstart[p + 1]; ++zp) {
          if (t.op_a[zp] != ap) continue;
          for (int zq = t.opstart[q]; zq < t.opstart[q + 1]; ++zq)
            if (t.op_c[zq] == cp)
              s += t.op_x[zp] * t.op_x[zq] * V.E(p + 1, q - 1, t.op_c[zp], t.op_a[zq]) * cm.wtm[P][t.op_b[zp]][t.op_b[zq]];
        }
        return w0 * wh * s;
      });
      // one-inner-pair terms are numbered by total size tt = l1 + l2 ascending, then l1 ascending
      int tmax = min(maxint, d - 2 - mh1);
      const int nterm = tmax >= 0 ? (tmax + 1) * (tmax + 2) / 2 : 0;
      auto term_l1l2 = [&](int term, int& l1, int& l2) {
        int tt = (int)((sqrt(8.0 * term + 1.0) - 1.0) * 0.5);
        while ((tt + 1) * (tt + 2) / 2 <= term) ++tt;
        while (tt * (tt + 1) / 2 > term) --tt;
        l1 = term - tt * (tt + 1) / 2;
        l2 = tt - l1;
      };
      auto loopw = [&](int term, int pz) {
        int ap, cp, l1, l2;
        const double w0 = zw(pz, ap, cp);
        if (w0 == 0.0) return 0.0;
        term_l1l2(term, l1, l2);
        return w0 * iloop_total(V, i, j, p + l1, q - l2, P, ap, cp);
      };
      // segment 1: stack (term 0), per (z_i,z_j)
      const int base1 = npair, n1 = nterm > 0 ? npair : 0;
      if (!done && n1 > 0) done = scan_segment(lane, pk, base1, n1, [&](int pz) { return loopw(0, pz); });
      // segment 2: multiloop, per (z_i,z_j) x bond index of the split (k asc, s asc)
      const int base2 = base1 + n1;
      const int kb0 = t.off[i + 2], kb1 = t.off[j];  // bonds of positions k = i+2 .. j-1
      const int nml = kb1 > kb0 ? kb1 - kb0 : 0;
      auto mlw = [&](int idx) {
        int ap, cp;
        const double w0 = zw(idx / nml, ap, cp);
        if (w0 == 0.0) return 0.0;
        const int kb = kb0 + idx % nml;
        return w0 * cm.wac * b.QM[(size_t)(t.off[p] + ap) * S + kb] * b.QM1T[(size_t)(t.off[q + 1] + cp) * S + kb];
      };
      // The segment's total is known in closed form (w_a w_c M2(p,q), stored by the inside pass): when the threshold lies
      // clearly beyond it, the O(d) scan over split points is skipped; within 1e-9 of its end it is scanned in order.
      bool skipped2 = false;
      double run2 = 0.0;
      int last2 = -1;
      if (!done && nml > 0) {
        const double tot2 = warp_total(lane, npair, [&](int pz) {
          int ap, cp;
          const double w0 = zw(pz, ap, cp);
          return w0 == 0.0 ? 0.0 : w0 * cm.wac * b.M2[(size_t)(t.off[p] + ap) * S + t.off[q + 1] + cp];
        });
        if (pk.thr > (pk.run + tot2) * (1.0 + 1e-9)) {
          skipped2 = true;
          run2 = pk.run;
          last2 = pk.last;
          pk.run += tot2;
          if (tot2 > 0.0) pk.last = base2 + npair * nml - 1;
        } else {
          done = scan_segment(lane, pk, base2, npair * nml, mlw);
        }
      }
      // segment 3: one inner pair with l1 + l2 >= 1, term outer, (z_i,z_j) inner
      const int base3 = base2 + npair * nml;
      if (!done && nterm > 1)
        done = scan_segment(lane, pk, base3, (nterm - 1) * npair,
                            [&](int idx) { return loopw(1 + idx / npair, idx % npair); });
      if (pk.hit < 0 && skipped2 && pk.last == base2 + npair * nml - 1) {
        // rounding left the threshold beyond every alternative and the last positive one is a split point: find it
        pk.run = run2;
        pk.last = last2;
        scan_segment(lane, pk, base2, npair * nml, mlw);
      }
      const int pick = pk.hit >= 0 ? pk.hit : pk.last;
      int ap, cp;
      if (pick < npair) {
        // hairpin: joint choice of the operators at p and q (K_HAIRPIN), then the interior chain
        zw(pick, ap, cp);
        const int zp0 = t.opstart[p], np = t.opstart[p + 1] - zp0, zq0 = t.opstart[q], nq = t.opstart[q + 1] - zq0;
        auto wf = [&](int k) {
          const int zp = zp0 + k / nq, zq = zq0 + k % nq;
          if (t.op_a[zp] != ap || t.op_c[zq] != cp) return 0.0;
          return t.op_x[zp] * t.op_x[zq] * V.E(p + 1, q - 1, t.op_c[zp], t.op_a[zq]) * cm.wtm[P][t.op_b[zp]][t.op_b[zq]];
        };
        Pick p2; p2.run = 0.0; p2.last = -1; p2.hit = -1;
        p2.thr = uniform(seed, smp, K_HAIRPIN, i, j) * warp_total(lane, np * nq, wf);
        scan_segment(lane, p2, 0, np * nq, wf);
        const int k = p2.hit >= 0 ? p2.hit : p2.last;
        const int zp = zp0 + k / nq, zq = zq0 + k % nq;
        if (lane == 0) { seq[p] = t.op_b[zp]; seq[q] = t.op_b[zq]; }
        chain(p + 1, q - 1, t.op_c[zp], t.op_a[zq]);
      } else if (pick >= base2 && pick < base3) {
        const int idx = pick - base2;
        zw(idx / nml, ap, cp);
        const int kb = kb0 + idx % nml;
        const int k = t.bondpos[kb], s = kb - t.off[k];
        if (lane == 0) {
          stk[sp] = Item{IT_QM, p, k - 1, (short)ap, 0, 0, (short)s};
          stk[sp + 1] = Item{IT_QM1, k, q, (short)s, 0, 0, (short)cp};
        }
        sp += 2;
      } else {
        int term, pz, l1, l2;
        if (pick < base2) { term = 0; pz = pick - base1; }
        else { term = 1 + (pick - base3) / npair; pz = (pick - base3) % npair; }
        zw(pz, ap, cp);
        term_l1l2(term, l1, l2);
        const int k = p + l1, l = q - l2;
        // level B (K_ILOOP): left side x right side x (x',y'), rectangular order
        // The left side runs over (operator at i+1) x (operator at k-1), the right side over (operator at l+1) x (operator at j-1); only the
        // operators at i+1 with a = ap and at j-1 with c = cp can weigh in, so those two lists are compacted (operator indices) and the
        // alternatives are numbered over the compact products, in the same order.
        short* lz = s_cz[wrp][0];
        short* rz = s_cz[wrp][1];
        const int zl0 = t.opstart[i + 1], nl1 = l1 >= 1 ? t.opstart[i + 2] - zl0 : 0, nl2 = l1 >= 2 ? t.opstart[k] - t.opstart[k - 1] : 1;
        const int zr0 = t.opstart[j - 1], nr2 = l2 >= 1 ? t.opstart[j] - zr0 : 0, nr1 = l2 >= 2 ? t.opstart[l + 2] - t.opstart[l + 1] : 1;
        int cl = 0, cr = 0;
        __syncwarp();
        for (int b0 = 0; b0 < nl1; b0 += 32) {
          const bool ok = b0 + lane < nl1 && t.op_a[zl0 + b0 + lane] == ap;
          const unsigned m = __ballot_sync(0xffffffffu, ok);
          const int pos = cl + __popc(m & ((1u << lane) - 1u));
          if (ok && pos < CCAP) lz[pos] = (short)(b0 + lane);
          cl += __popc(m);
        }
        for (int b0 = 0; b0 < nr2; b0 += 32) {
          const bool ok = b0 + lane < nr2 && t.op_c[zr0 + b0 + lane] == cp;
          const unsigned m = __ballot_sync(0xffffffffu, ok);
          const int pos = cr + __popc(m & ((1u << lane) - 1u));
          if (ok && pos < CCAP) rz[pos] = (short)(b0 + lane);
          cr += __popc(m);
        }
        __syncwarp();
        const bool cside = cl <= CCAP && cr <= CCAP;
        // compact side index -> index of the rectangular numbering of left_side / right_side
        auto lmap = [&](int la) { return (!cside || l1 == 0) ? la : l1 == 1 ? (int)lz[la] : lz[la / nl2] * nl2 + la % nl2; };
        auto rmap = [&](int ra) { return (!cside || l2 == 0) ? ra : l2 == 1 ? (int)rz[ra] : (ra / cr) * nr2 + rz[ra % cr]; };
        const int nl = (!cside || l1 == 0) ? left_count(t, i, k) : cl * nl2;
        const int nr = (!cside || l2 == 0) ? right_count(t, j, l) : nr1 * cr;
        auto wf = [&](int f) {
          const int xy = f & 15, ra = rmap((f >> 4) % nr), la = lmap((f >> 4) / nr);
          const int xp = xy >> 2, yp = xy & 3;
          if (!V.can(xp, yp)) return 0.0;
          const SideL L = left_side(V, i, k, ap, la);
          if (L.w == 0.0) return 0.0;
          const SideL R = right_side(V, j, l, cp, ra);
          if (R.w == 0.0) return 0.0;
          return loop_factor(V, P, l1, l2, xp, yp, L, R) * L.w * R.w * V.QB(k, l, L.s, xp, yp, R.s);
        };
        Pick p2; p2.run = 0.0; p2.last = -1; p2.hit = -1;
        p2.thr = uniform(seed, smp, K_ILOOP, i, j) * warp_total(lane, nl * nr * 16, wf);
        scan_segment(lane, p2, 0, nl * nr * 16, wf);
        const int f = p2.hit >= 0 ? p2.hit : p2.last;
        const int xy = f & 15, ra = rmap((f >> 4) % nr), la = lmap((f >> 4) / nr);
        const SideL L = left_side(V, i, k, ap, la);
        const SideL R = right_side(V, j, l, cp, ra);
        if (l1 >= 1 && lane == 0) seq[i + 1] = (uint8_t)L.u;
        if (l1 >= 2) {
          if (lane == 0) seq[k - 1] = (uint8_t)L.up;
          chain(i + 2, k - 2, t.op_c[L.z1], t.op_a[L.z2]);
        }
        if (l2 >= 1 && lane == 0) seq[j - 1] = (uint8_t)R.u;
        if (l2 >= 2) {
          if (lane == 0) seq[l + 1] = (uint8_t)R.up;
          chain(l + 2, j - 2, t.op_c[R.z1], t.op_a[R.z2]);
        }
        if (lane == 0) stk[sp] = Item{IT_QB, k, l, (short)L.s, (short)(xy >> 2), (short)(xy & 3), (short)R.s};
        ++sp;
      }
    }
    __syncwarp();
  }
}

}  // namespace

int cdz_launch_sample(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, cudaStream_t st) {
  const int cap = t->tt->n / 4 + 16;
  Item* stacks = nullptr;
  CDZ_CUDA(cudaMallocAsync((void**)&stacks, sizeof(Item) * (size_t)cap * J, st));
  const int wpb = 4;
  t->launches[5] = 1;
  if (t->ev_class.size() > t->nev_inside) t->ev_class.resize(t->nev_inside);  // one traceback's events after the pass's, not a growing list
  auto mark = [&](int cls) {
    if (!t->profile) return;
    const size_t k = t->ev_class.size();
    if (k >= t->evs.size()) { cudaEvent_t e; cudaEventCreate(&e); t->evs.push_back(e); }
    cudaEventRecord(t->evs[k], st);
    t->ev_class.push_back(cls);
  };
  mark(5);
  sample_kernel<<<(J + wpb - 1) / wpb, wpb * 32, 0, st>>>(t->d_ctx, J, seed, seq_dev, pair_dev, stacks, cap);
  mark(7);
  CDZ_CUDA(cudaGetLastError());
  CDZ_CUDA(cudaFreeAsync(stacks, st));
  return CDZ_OK;
}

// ------------------------------------------------------------------------------------------------
// cdz_sample_noalloc: the same traceback for callers that cannot allocate device memory (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The per-sample decision stacks -- the only scratch sample_kernel needs -- live in a
// file-scope device array instead of a stream-ordered allocation.  Every GPU that loads the library holds the array
// (CDZ_NOALLOC_STACK_ITEMS x 20 bytes = 8.0 MB) until the process exits; every call on a device shares it, so calls that overlap
// on one GPU race.  Nothing in it has to start at zero: a warp pushes an item before it pops it.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) Item g_noalloc_stacks[CDZ_NOALLOC_STACK_ITEMS];

namespace {
constexpr int NOALLOC_MAX_DEV = 64;
Item* g_noalloc_ptr[NOALLOC_MAX_DEV];  // device address of g_noalloc_stacks, per device (the symbol itself is only a host-side stand-in)
std::mutex g_noalloc_mu;
}  // namespace

extern "C" int cdz_sample_noalloc(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, void* stream) {
  static_assert(sizeof(Item) == 20, "cdz.h documents 20 bytes per stack item");
  if (!t || J < 0 || !seq_dev || !pair_dev) { cdz_set_error("cdz_sample_noalloc: bad argument"); return CDZ_EINVAL; }
  if (!t->done) { cdz_set_error("cdz_sample_noalloc before cdz_inside"); return CDZ_ESTATE; }
  if (J == 0) return CDZ_OK;
  const int cap = t->tt->n / 4 + 16;  // stack depth per sample, as in cdz_sample
  if ((long long)cap * J > (long long)CDZ_NOALLOC_STACK_ITEMS) {
    char msg[256];
    snprintf(msg, sizeof(msg), "cdz_sample_noalloc: J x (n/4 + 16) = %d x %d stack items exceed the static scratch of %d items (J <= %d at n = %d); "
             "use cdz_sample", J, cap, CDZ_NOALLOC_STACK_ITEMS, CDZ_NOALLOC_STACK_ITEMS / cap, t->tt->n);
    cdz_set_error(msg);
    return CDZ_EINVAL;
  }
  int dev = -1;
  CDZ_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEV) { cdz_set_error("cdz_sample_noalloc: device ordinal beyond 63"); return CDZ_EINVAL; }
  Item* stacks = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {  // once per device, with that device current
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_noalloc_stacks) != cudaSuccess || !p) {
        cudaGetLastError();
        cdz_set_error("cdz_sample_noalloc: cudaGetSymbolAddress of the static scratch failed");
        return CDZ_ECUDA;
      }
      g_noalloc_ptr[dev] = (Item*)p;
    }
    stacks = g_noalloc_ptr[dev];
  }
  cudaStream_t st = (cudaStream_t)stream;
  const int rc = cdz_wait_pass(t, st);
  if (rc != CDZ_OK) return rc;
  const int wpb = 4;
  sample_kernel<<<(J + wpb - 1) / wpb, wpb * 32, 0, st>>>(t->d_ctx, J, seed, seq_dev, pair_dev, stacks, cap);
  CDZ_CUDA(cudaGetLastError());
  return CDZ_OK;
}
