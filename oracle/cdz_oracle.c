/*
 * cdz_oracle.c -- CPU ORACLE (test infrastructure, NOT the product; see cdz_oracle.h).
 *
 * Everything here is written for legibility against PAPER.md and DESIGN.md, in
 * long double, with no blocking / fusion / scaling tricks.  Unscaled long double
 * holds e^{+-11356}, i.e. log Z up to ~1.1e4, enough for n <= ~8000 nt with the
 * synthetic model (log Z ~ 1.33 nat/nt); larger designs are checked window-wise.
 */
#include "cdz_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double real;

struct orc_tt {
  int n;
  int* sigma; /* [n+1] bond dimensions, sigma[0] must be 1 */
  int* start; /* [n+1] operator list offsets */
  orc_op* ops;
};

/* ------------------------------------------------------------------------- */
/* genetic code, codon index = 16 b0 + 4 b1 + b2 with A,C,G,U = 0..3           */
/* (the sense codons per amino acid are those listed in PAPER.md lines 859-881) */
/* ------------------------------------------------------------------------- */
static const char GENETIC_CODE[65] =
    "KNKNTTTTRSRSIIMI"
    "QHQHPPPPRRRRLLLL"
    "EDEDAAAAGGGGVVVV"
    "*Y*YSSSS*CWCLFLF";

static int codons_of(char aa, int* out) {
  int k = 0;
  for (int c = 0; c < 64; ++c)
    if (GENETIC_CODE[c] == aa && aa != '*') out[k++] = c;
  return k;
}

static int rank_in(const int* set, int count, int v) {
  for (int r = 0; r < count; ++r)
    if (set[r] == v) return r;
  return -1;
}

/* distinct values of base `pos` (0,1,2) among codons, ascending */
static int distinct_bases(const int* cod, int deg, int pos, int* out) {
  int k = 0;
  for (int b = 0; b < 4; ++b)
    for (int t = 0; t < deg; ++t) {
      int cb = (cod[t] >> (2 * (2 - pos))) & 3;
      if (cb == b) { out[k++] = b; break; }
    }
  return k;
}

/* cw_stride = 0: one codon table [64] for all residues; 64: one table per residue, codon_logw[L][64] (PAPER.md line 157:
 * the soft constraint penalises codon c "at amino acid position i") */
static int tt_build_impl(const char* aa, int L, int kind, const double* codon_logw, int cw_stride, const double* pair_logw,
                         orc_tt** out) {
  if (L <= 0 || !aa || !out) return -1;
  int n = 3 * L;
  orc_tt* tt = (orc_tt*)calloc(1, sizeof(orc_tt));
  tt->n = n;
  tt->sigma = (int*)calloc(n + 1, sizeof(int));
  tt->start = (int*)calloc(n + 1, sizeof(int));
  tt->ops = (orc_op*)calloc((size_t)L * 48 + 8, sizeof(orc_op));
  int nops = 0;
  int prev[6], pdeg = 1;
  prev[0] = -1; /* fictitious one-codon predecessor */
  for (int k = 0; k < L; ++k) {
    int cod[6];
    int deg = codons_of(aa[k], cod);
    if (deg == 0) { orc_tt_free(tt); return -2; }
    if (kind == 0) {
      /* single-codon TT: eq 3.4 (line 151), operator lists S3c.i (lines 559-563) */
      int fb[4], tb[4];
      int nf = distinct_bases(cod, deg, 0, fb), nt = distinct_bases(cod, deg, 2, tb);
      tt->sigma[3 * k] = 1;
      tt->sigma[3 * k + 1] = nf;
      tt->sigma[3 * k + 2] = nt;
      tt->start[3 * k] = nops;
      for (int r = 0; r < nf; ++r) tt->ops[nops++] = (orc_op){0, fb[r], r, 1.0};
      tt->start[3 * k + 1] = nops;
      for (int t = 0; t < deg; ++t) {
        int b0 = cod[t] >> 4, b1 = (cod[t] >> 2) & 3, b2 = cod[t] & 3;
        double x = codon_logw ? exp(codon_logw[(size_t)k * cw_stride + cod[t]]) : 1.0; /* line 157 */
        tt->ops[nops++] = (orc_op){rank_in(fb, nf, b0), b1, rank_in(tb, nt, b2), x};
      }
      tt->start[3 * k + 2] = nops;
      for (int r = 0; r < nt; ++r) tt->ops[nops++] = (orc_op){r, tb[r], 0, 1.0};
    } else {
      /* codon-pair TT: eq 3.3 (line 145) in the S3c.ii form (lines 565-569):
       * transition + pair weight on the 5' base, codon weight on the middle base */
      tt->sigma[3 * k] = pdeg;
      tt->sigma[3 * k + 1] = deg;
      tt->sigma[3 * k + 2] = deg;
      tt->start[3 * k] = nops;
      for (int a = 0; a < pdeg; ++a)
        for (int c = 0; c < deg; ++c) {
          double x = (k > 0 && pair_logw) ? exp(pair_logw[prev[a] * 64 + cod[c]]) : 1.0; /* line 163 */
          tt->ops[nops++] = (orc_op){a, cod[c] >> 4, c, x};
        }
      tt->start[3 * k + 1] = nops;
      for (int c = 0; c < deg; ++c) {
        double x = codon_logw ? exp(codon_logw[(size_t)k * cw_stride + cod[c]]) : 1.0;
        tt->ops[nops++] = (orc_op){c, (cod[c] >> 2) & 3, c, x};
      }
      tt->start[3 * k + 2] = nops;
      for (int c = 0; c < deg; ++c) tt->ops[nops++] = (orc_op){c, cod[c] & 3, c, 1.0};
      memcpy(prev, cod, sizeof(cod));
      pdeg = deg;
    }
  }
  tt->start[n] = nops;
  tt->sigma[n] = (kind == 0) ? 1 : pdeg;
  *out = tt;
  return 0;
}

int orc_tt_build(const char* aa, int L, int kind, const double* codon_logw, const double* pair_logw, orc_tt** out) {
  return tt_build_impl(aa, L, kind, codon_logw, 0, pair_logw, out);
}
int orc_tt_build_pos(const char* aa, int L, int kind, const double* codon_logw_pos, const double* pair_logw, orc_tt** out) {
  return tt_build_impl(aa, L, kind, codon_logw_pos, 64, pair_logw, out);
}

int orc_tt_from_ops(int n, const int* counts, const orc_op* ops, orc_tt** out) {
  if (n <= 0) return -1;
  orc_tt* tt = (orc_tt*)calloc(1, sizeof(orc_tt));
  tt->n = n;
  tt->sigma = (int*)calloc(n + 1, sizeof(int));
  tt->start = (int*)calloc(n + 1, sizeof(int));
  int tot = 0;
  for (int i = 0; i < n; ++i) { tt->start[i] = tot; tot += counts[i]; }
  tt->start[n] = tot;
  tt->ops = (orc_op*)calloc(tot + 1, sizeof(orc_op));
  memcpy(tt->ops, ops, sizeof(orc_op) * tot);
  for (int i = 0; i <= n; ++i) tt->sigma[i] = 1;
  for (int i = 0; i < n; ++i)
    for (int z = tt->start[i]; z < tt->start[i + 1]; ++z) {
      if (ops[z].a + 1 > tt->sigma[i]) tt->sigma[i] = ops[z].a + 1;
      if (ops[z].c + 1 > tt->sigma[i + 1]) tt->sigma[i + 1] = ops[z].c + 1;
    }
  *out = tt;
  return 0;
}

void orc_tt_free(orc_tt* tt) {
  if (!tt) return;
  free(tt->sigma); free(tt->start); free(tt->ops); free(tt);
}
int orc_tt_n(const orc_tt* tt) { return tt->n; }
int orc_tt_nops(const orc_tt* tt) { return tt->start[tt->n]; }
void orc_tt_get(const orc_tt* tt, int* sigma, int* counts, orc_op* ops) {
  if (sigma) memcpy(sigma, tt->sigma, sizeof(int) * (tt->n + 1));
  if (counts) for (int i = 0; i < tt->n; ++i) counts[i] = tt->start[i + 1] - tt->start[i];
  if (ops) memcpy(ops, tt->ops, sizeof(orc_op) * tt->start[tt->n]);
}

/* eq 3.2, open chain: e_0^T Tbar_0 ... Tbar_{n-1} 1 */
double orc_tt_logsum(const orc_tt* tt) {
  int maxs = 1;
  for (int i = 0; i <= tt->n; ++i) if (tt->sigma[i] > maxs) maxs = tt->sigma[i];
  real* v = (real*)calloc(maxs, sizeof(real));
  real* w = (real*)calloc(maxs, sizeof(real));
  v[0] = 1.0L;
  for (int i = 0; i < tt->n; ++i) {
    for (int c = 0; c < maxs; ++c) w[c] = 0;
    for (int z = tt->start[i]; z < tt->start[i + 1]; ++z) w[tt->ops[z].c] += v[tt->ops[z].a] * (real)tt->ops[z].x;
    memcpy(v, w, sizeof(real) * maxs);
  }
  real s = 0;
  for (int c = 0; c < tt->sigma[tt->n]; ++c) s += v[c];
  free(v); free(w);
  return (double)logl(s);
}

/* ------------------------------------------------------------------------- */
/* energy model                                                              */
/* ------------------------------------------------------------------------- */
static const int PTYPE[4][4] = {
    /* A */ {-1, -1, -1, 0},
    /* C */ {-1, -1, 1, -1},
    /* G */ {-1, 2, -1, 4},
    /* U */ {3, -1, 5, -1}};

static double model_kT(const orc_model* m) { return (8.31446261815324 / 4184.0) * m->temperature_K; }

static int can_pair(const orc_model* m, int x, int y) { return m->allow_all_pairs || PTYPE[x][y] >= 0; }
static int ptype(int x, int y) { return PTYPE[x][y] >= 0 ? PTYPE[x][y] : 0; }

static double hairpin_init(const orc_model* m, int l) {
  return m->hairpin_a + m->hairpin_b * model_kT(m) * log((double)l / m->hairpin_l0);
}

/* E(phi,s): sum over loops of the nearest-neighbour decomposition */
double orc_energy(const orc_model* m, int n, const uint8_t* seq, const int32_t* pair, int* valid) {
  double E = 0.0;
  *valid = 1;
  for (int i = 0; i < n; ++i) {
    int j = pair[i];
    if (j < 0) continue;
    if (j >= n || pair[j] != i || j == i) { *valid = 0; return 0; }
    if (j < i) continue;
    if (!can_pair(m, seq[i], seq[j])) { *valid = 0; return 0; }
    /* loop closed by (i,j): scan its interior */
    int branches = 0, unpaired = 0, k1 = -1, l1p = -1;
    for (int p = i + 1; p < j;) {
      if (pair[p] < 0) { ++unpaired; ++p; continue; }
      if (pair[p] < p || pair[p] > j) { *valid = 0; return 0; } /* crossing */
      if (branches == 0) { k1 = p; l1p = pair[p]; }
      ++branches;
      p = pair[p] + 1;
    }
    int P = ptype(seq[i], seq[j]);
    if (branches == 0) {
      int l = j - i - 1;
      if (l < m->min_hairpin) { *valid = 0; return 0; }
      E += hairpin_init(m, l) + m->tmm[P][seq[i + 1]][seq[j - 1]];
    } else if (branches == 1) {
      int la = k1 - i - 1, lb = j - l1p - 1;
      int Pin = ptype(seq[k1], seq[l1p]);
      if (la + lb > m->max_interior) { *valid = 0; return 0; }
      if (la == 0 && lb == 0) {
        E += m->stack[P][Pin];
      } else if (la == 0 || lb == 0) {
        int l = la + lb;
        E += m->bulge_init[l] + (l == 1 ? m->stack[P][Pin] : 0.0);
      } else {
        E += m->interior_init[la + lb] + m->tmm[P][seq[i + 1]][seq[j - 1]] +
             m->tmm[ptype(seq[l1p], seq[k1])][seq[l1p + 1]][seq[k1 - 1]];
      }
    } else {
      E += m->ml_a + m->ml_c * (branches + 1) + m->ml_b * unpaired;
    }
  }
  return E;
}

/* W(phi): e_0^T prod_i T_i^{phi_i} 1 (eq 3.1 with open boundaries) */
static real tt_seq_weight(const orc_tt* tt, const uint8_t* seq) {
  int maxs = 1;
  for (int i = 0; i <= tt->n; ++i) if (tt->sigma[i] > maxs) maxs = tt->sigma[i];
  real v[64], w[64];
  if (maxs > 64) return 0;
  for (int c = 0; c < maxs; ++c) v[c] = 0;
  v[0] = 1;
  for (int i = 0; i < tt->n; ++i) {
    for (int c = 0; c < maxs; ++c) w[c] = 0;
    for (int z = tt->start[i]; z < tt->start[i + 1]; ++z)
      if (tt->ops[z].b == seq[i]) w[tt->ops[z].c] += v[tt->ops[z].a] * (real)tt->ops[z].x;
    memcpy(v, w, sizeof(real) * maxs);
  }
  real s = 0;
  for (int c = 0; c < tt->sigma[tt->n]; ++c) s += v[c];
  return s;
}

double orc_logweight(const orc_model* m, const orc_tt* tt, const uint8_t* seq, const int32_t* pair) {
  int valid;
  double E = orc_energy(m, tt->n, seq, pair, &valid);
  real W = tt_seq_weight(tt, seq);
  if (!valid || W <= 0) return -INFINITY;
  return (double)(logl(W) - (real)(E / model_kT(m)));
}

/* ---- brute force: enumerate operator paths x structures -------------------- */
typedef struct {
  const orc_model* m;
  const orc_tt* tt;
  int n;
  uint8_t* seq;
  int32_t* pair;
  int* stack; /* open right ends */
  int sp;
  real W;     /* weight of current sequence */
  real Z;
  real* bpp; real* base; real* codon;
  double nstates;
  double beta;
} bf_ctx;

static void bf_structures(bf_ctx* c, int i) {
  int n = c->n;
  if (i == n) {
    int valid;
    double E = orc_energy(c->m, n, c->seq, c->pair, &valid);
    if (!valid) return;
    real w = c->W * expl(-(real)E * (real)c->beta);
    c->Z += w;
    c->nstates += 1.0;
    if (c->bpp)
      for (int p = 0; p < n; ++p) {
        if (c->pair[p] < 0) c->bpp[p * n + p] += w;
        else if (c->pair[p] > p) c->bpp[p * n + c->pair[p]] += w;
      }
    if (c->base) for (int p = 0; p < n; ++p) c->base[p * 4 + c->seq[p]] += w;
    if (c->codon)
      for (int k = 0; k < n / 3; ++k)
        c->codon[k * 64 + 16 * c->seq[3 * k] + 4 * c->seq[3 * k + 1] + c->seq[3 * k + 2]] += w;
    return;
  }
  if (c->sp > 0 && c->stack[c->sp - 1] == i) { /* i closes the innermost open pair */
    --c->sp;
    bf_structures(c, i + 1);
    c->stack[c->sp++] = i;
    return;
  }
  c->pair[i] = -1;
  bf_structures(c, i + 1);
  int lim = c->sp > 0 ? c->stack[c->sp - 1] : n;
  for (int j = i + c->m->min_hairpin + 1; j < lim; ++j) {
    if (!can_pair(c->m, c->seq[i], c->seq[j])) continue;
    c->pair[i] = j; c->pair[j] = i;
    c->stack[c->sp++] = j;
    bf_structures(c, i + 1);
    --c->sp;
    c->pair[i] = -1; c->pair[j] = -1;
  }
}

static void bf_sequences(bf_ctx* c, int i, int bond, real W) {
  if (i == c->n) {
    c->W = W;
    for (int p = 0; p < c->n; ++p) c->pair[p] = -1;
    c->sp = 0;
    bf_structures(c, 0);
    return;
  }
  for (int z = c->tt->start[i]; z < c->tt->start[i + 1]; ++z) {
    const orc_op* o = &c->tt->ops[z];
    if (o->a != bond) continue;
    c->seq[i] = (uint8_t)o->b;
    bf_sequences(c, i + 1, o->c, W * (real)o->x);
  }
}

int orc_brute_force(const orc_model* m, const orc_tt* tt, double* logZ, double* bpp, double* base,
                    double* codon, double* n_states) {
  int n = tt->n;
  bf_ctx c;
  memset(&c, 0, sizeof(c));
  c.m = m; c.tt = tt; c.n = n;
  c.seq = (uint8_t*)calloc(n, 1);
  c.pair = (int32_t*)calloc(n, sizeof(int32_t));
  c.stack = (int*)calloc(n + 1, sizeof(int));
  c.beta = 1.0 / model_kT(m);
  if (bpp) c.bpp = (real*)calloc((size_t)n * n, sizeof(real));
  if (base) c.base = (real*)calloc((size_t)n * 4, sizeof(real));
  if (codon) c.codon = (real*)calloc((size_t)(n / 3) * 64, sizeof(real));
  bf_sequences(&c, 0, 0, 1.0L);
  if (logZ) *logZ = (double)logl(c.Z);
  if (n_states) *n_states = c.nstates;
  if (bpp) { for (int p = 0; p < n * n; ++p) bpp[p] = (double)(c.bpp[p] / c.Z); free(c.bpp); }
  if (base) { for (int p = 0; p < n * 4; ++p) base[p] = (double)(c.base[p] / c.Z); free(c.base); }
  if (codon) { for (int p = 0; p < (n / 3) * 64; ++p) codon[p] = (double)(c.codon[p] / c.Z); free(c.codon); }
  free(c.seq); free(c.pair); free(c.stack);
  return 0;
}

double orc_count_structures(int n, int min_hairpin, int max_interior) {
  orc_model m;
  memset(&m, 0, sizeof(m));
  m.temperature_K = 310.15;
  m.hairpin_l0 = 1.0;
  m.max_interior = max_interior;
  m.min_hairpin = min_hairpin;
  m.allow_all_pairs = 1;
  int* counts = (int*)calloc(n, sizeof(int));
  orc_op* ops = (orc_op*)calloc(n, sizeof(orc_op));
  for (int i = 0; i < n; ++i) { counts[i] = 1; ops[i] = (orc_op){0, 0, 0, 1.0}; }
  orc_tt* tt;
  orc_tt_from_ops(n, counts, ops, &tt);
  double ns = 0;
  orc_brute_force(&m, tt, NULL, NULL, NULL, NULL, &ns);
  orc_tt_free(tt); free(counts); free(ops);
  return ns;
}

/* ---- scalar fixed-sequence McCaskill, textbook decomposition ----------------
 * Q(i,j)  : all structures on [i..j]            (exterior, energy 0)
 * Qb(i,j) : i.j paired
 * Qm(i,j) : >=1 branch inside a multiloop,  Qm = sum_k [w_b^{k-i} + Qm(i,k-1)] Qm1(k,j)
 * Qm1(i,j): exactly one branch starting at i, trailing unpaired.
 * Deliberately a different decomposition from the tensor recursion below.       */
double orc_mccaskill(const orc_model* m, int n, const uint8_t* seq) {
  double beta = 1.0 / model_kT(m);
#define IX(i, j) ((size_t)(i) * n + (j))
  real* Q = (real*)calloc((size_t)n * n, sizeof(real));
  real* Qb = (real*)calloc((size_t)n * n, sizeof(real));
  real* Qm = (real*)calloc((size_t)n * n, sizeof(real));
  real* Qm1 = (real*)calloc((size_t)n * n, sizeof(real));
  real wa = expl(-(real)(m->ml_a * beta)), wb = expl(-(real)(m->ml_b * beta)), wc = expl(-(real)(m->ml_c * beta));
  for (int d = 0; d < n; ++d)
    for (int i = 0; i + d < n; ++i) {
      int j = i + d;
      real qb = 0;
      if (d >= m->min_hairpin + 1 && can_pair(m, seq[i], seq[j])) {
        int P = ptype(seq[i], seq[j]);
        qb += expl(-(real)((hairpin_init(m, d - 1) + m->tmm[P][seq[i + 1]][seq[j - 1]]) * beta));
        for (int k = i + 1; k < j; ++k)
          for (int l = j - 1; l > k; --l) {
            int la = k - i - 1, lb = j - l - 1;
            if (la + lb > m->max_interior) break;
            if (Qb[IX(k, l)] == 0) continue;
            int Pin = ptype(seq[k], seq[l]);
            double e;
            if (la == 0 && lb == 0) e = m->stack[P][Pin];
            else if (la == 0 || lb == 0) e = m->bulge_init[la + lb] + (la + lb == 1 ? m->stack[P][Pin] : 0.0);
            else e = m->interior_init[la + lb] + m->tmm[P][seq[i + 1]][seq[j - 1]] +
                     m->tmm[ptype(seq[l], seq[k])][seq[l + 1]][seq[k - 1]];
            qb += expl(-(real)(e * beta)) * Qb[IX(k, l)];
          }
        /* multiloop: at least two branches in [i+1..j-1] */
        for (int k = i + 2; k <= j - 1; ++k)
          qb += wa * wc * Qm[IX(i + 1, k - 1)] * Qm1[IX(k, j - 1)];
      }
      Qb[IX(i, j)] = qb;
      Qm1[IX(i, j)] = wc * qb + (j > i ? wb * Qm1[IX(i, j - 1)] : 0);
      real qm = 0, wlead = 1;
      for (int k = i; k <= j; ++k) {
        qm += (wlead + (k > i ? Qm[IX(i, k - 1)] : 0)) * Qm1[IX(k, j)];
        wlead *= wb;
      }
      Qm[IX(i, j)] = qm;
      /* exterior: j unpaired, or j pairs with k */
      real q = (j > i ? Q[IX(i, j - 1)] : 1.0L);
      for (int k = i; k <= j; ++k) q += (k > i ? Q[IX(i, k - 1)] : 1.0L) * Qb[IX(k, j)];
      Q[IX(i, j)] = q;
    }
  double r = (double)logl(Q[IX(0, n - 1)]);
  free(Q); free(Qb); free(Qm); free(Qm1);
#undef IX
  return r;
}

/* ------------------------------------------------------------------------- */
/* tensor-valued inside recursion */
/* ------------------------------------------------------------------------- */
struct orc_tables {
  int n;
  orc_tt* tt; /* private copy */
  orc_model model;
  int* sig;
  real** Td; /* Td[i][(a*4+x)*sig[i+1]+c]  = T_i[a,x,c]  (eq S3.7) */
  real** Tb; /* Tb[i][a*sig[i+1]+c]        = Tbar_i      (line 135) */
  real** E;  /* E(i,j) = Tbar_i..Tbar_j, index i*(n+1)+(j+1), j >= i-1 (identity) */
  real **qb, **qbs, **qm1, **qml, **m2, **qm; /* index i*n+j */
  real** qext; /* qext[j+1][c], qext[0] = [1] */
  real wst[6][6], wtm[6][4][4], wbu[31], win[31], wa, wb, wc;
  double beta;
  int forbid_i, forbid_j; /* pair excluded from every structure (-1: none); used by orc_marginals */
};

#define SG(t, i) ((t)->sig[i])
static real* cell_alloc(size_t k) { return (real*)calloc(k ? k : 1, sizeof(real)); }

static const real* getE(const orc_tables* t, int i, int j) { return t->E[(size_t)i * (t->n + 1) + (j + 1)]; }

/* Up(p,q)[a,u,v,c] = sum T_p[a,u,.] E(p+1,q-1) T_q[.,v,c]  (p<q);  Up(p,p)[a,u,v,c] = delta_uv T_p[a,u,c] */
static void compute_Up(const orc_tables* t, int p, int q, real* out) {
  int Sa = SG(t, p), Sc = SG(t, q + 1);
  for (int k = 0; k < Sa * 16 * Sc; ++k) out[k] = 0;
  const orc_tt* tt = t->tt;
  if (p == q) {
    for (int z = tt->start[p]; z < tt->start[p + 1]; ++z) {
      const orc_op* o = &tt->ops[z];
      out[((o->a * 4 + o->b) * 4 + o->b) * Sc + o->c] += (real)o->x;
    }
    return;
  }
  const real* Em = getE(t, p + 1, q - 1);
  int Sm = SG(t, q); /* columns of E(p+1,q-1) */
  for (int z = tt->start[p]; z < tt->start[p + 1]; ++z)
    for (int y = tt->start[q]; y < tt->start[q + 1]; ++y) {
      const orc_op *o = &tt->ops[z], *r = &tt->ops[y];
      out[((o->a * 4 + o->b) * 4 + r->b) * Sc + r->c] += (real)o->x * Em[o->c * Sm + r->a] * (real)r->x;
    }
}

/* one closed cell: Qb(i,j)[a,x,y,c] following SURVEY App. A.2 term by term */
static void compute_qb(orc_tables* t, int i, int j) {
  const orc_model* m = &t->model;
  int n = t->n, d = j - i;
  int Si = SG(t, i), Sj1 = SG(t, j + 1);
  real* qb = t->qb[(size_t)i * n + j];
  if (d < m->min_hairpin + 1) return;
  if (i == t->forbid_i && j == t->forbid_j) return; /* restricted ensemble without the pair (i,j) */
  int Sa = SG(t, i + 1), Sc = SG(t, j); /* a' in Sigma_{i+1}, c' in Sigma_j */
  /* inner[x][y][a'][c'] */
  real* inner = cell_alloc((size_t)16 * Sa * Sc);
#define INNER(x, y, a, c) inner[(((x) * 4 + (y)) * Sa + (a)) * Sc + (c)]
  int maxS = 1;
  for (int p = i; p <= j + 1; ++p) if (SG(t, p) > maxS) maxS = SG(t, p);
  real* UpL = cell_alloc((size_t)maxS * 16 * maxS);
  real* UpR = cell_alloc((size_t)maxS * 16 * maxS);
  real* A1 = cell_alloc((size_t)maxS * 16 * 16 * maxS); /* [a'][u][u'][x'][y'][t] */
  real* A2 = cell_alloc((size_t)maxS * 16 * maxS);      /* [a'][u][v'][t] */
  real* A3 = cell_alloc((size_t)maxS * 16 * maxS);      /* [a'][u][v][c'] */

  /* hairpin: sum_{u,v} exp(-beta(H(d-1)+tmm[p(x,y)][u][v])) Up(i+1,j-1)[a',u,v,c'] */
  {
    compute_Up(t, i + 1, j - 1, UpL);
    real wh = expl(-(real)(hairpin_init(m, d - 1) * t->beta));
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        int P = ptype(x, y);
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int v = 0; v < 4; ++v)
              for (int c = 0; c < Sc; ++c)
                INNER(x, y, a, c) += wh * t->wtm[P][u][v] * UpL[((a * 4 + u) * 4 + v) * Sc + c];
      }
  }
  /* one inner pair (k,l): k ascending, l descending */
  for (int k = i + 1; k < j; ++k)
    for (int l = j - 1; l > k; --l) {
      int l1 = k - i - 1, l2 = j - l - 1;
      if (l1 + l2 > m->max_interior) break;
      if (l - k < m->min_hairpin + 1) continue;
      const real* qin = t->qb[(size_t)k * n + l]; /* [s][x'][y'][tt] */
      int Ss = SG(t, k), St = SG(t, l + 1);
      if (l1 == 0 && l2 == 0) {
        /* stack: Ss == Sa, St == Sc */
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            for (int xp = 0; xp < 4; ++xp)
              for (int yp = 0; yp < 4; ++yp) {
                if (!can_pair(m, xp, yp)) continue;
                real w = t->wst[ptype(x, y)][ptype(xp, yp)];
                for (int a = 0; a < Sa; ++a)
                  for (int c = 0; c < Sc; ++c) INNER(x, y, a, c) += w * qin[((a * 4 + xp) * 4 + yp) * St + c];
              }
          }
      } else if (l2 == 0) {
        /* left bulge: sum_s E(i+1,k-1)[a',s] Qb(k,l)[s,x',y',c'] */
        const real* El = getE(t, i + 1, k - 1);
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            for (int xp = 0; xp < 4; ++xp)
              for (int yp = 0; yp < 4; ++yp) {
                if (!can_pair(m, xp, yp)) continue;
                real w = t->wbu[l1] * (l1 == 1 ? t->wst[ptype(x, y)][ptype(xp, yp)] : 1.0L);
                for (int a = 0; a < Sa; ++a)
                  for (int s = 0; s < Ss; ++s)
                    for (int c = 0; c < Sc; ++c)
                      INNER(x, y, a, c) += w * El[a * Ss + s] * qin[((s * 4 + xp) * 4 + yp) * St + c];
              }
          }
      } else if (l1 == 0) {
        /* right bulge: sum_t Qb(k,l)[a',x',y',t] E(l+1,j-1)[t,c'] */
        const real* Er = getE(t, l + 1, j - 1);
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            for (int xp = 0; xp < 4; ++xp)
              for (int yp = 0; yp < 4; ++yp) {
                if (!can_pair(m, xp, yp)) continue;
                real w = t->wbu[l2] * (l2 == 1 ? t->wst[ptype(x, y)][ptype(xp, yp)] : 1.0L);
                for (int a = 0; a < Sa; ++a)
                  for (int tt_ = 0; tt_ < St; ++tt_)
                    for (int c = 0; c < Sc; ++c)
                      INNER(x, y, a, c) += w * qin[((a * 4 + xp) * 4 + yp) * St + tt_] * Er[tt_ * Sc + c];
              }
          }
      } else {
        /* generic interior loop, contracted in four explicit stages:
         *  sum exp(-beta(In(l1+l2)+tmm[p(x,y)][u][v]+tmm[p(y',x')][v'][u']))
         *      Up(i+1,k-1)[a',u,u',s] Qb(k,l)[s,x',y',t] Up(l+1,j-1)[t,v',v,c']        */
        compute_Up(t, i + 1, k - 1, UpL); /* [a'][u][u'][s]  */
        compute_Up(t, l + 1, j - 1, UpR); /* [t][v'][v][c']  */
        for (int q = 0; q < Sa * 16 * 16 * St; ++q) A1[q] = 0;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int up = 0; up < 4; ++up)
              for (int s = 0; s < Ss; ++s) {
                real w = UpL[((a * 4 + u) * 4 + up) * Ss + s];
                if (w == 0) continue;
                for (int xy = 0; xy < 16; ++xy)
                  for (int tt_ = 0; tt_ < St; ++tt_)
                    A1[((((a * 4 + u) * 4 + up) * 16) + xy) * St + tt_] += w * qin[(s * 16 + xy) * St + tt_];
              }
        for (int q = 0; q < Sa * 16 * St; ++q) A2[q] = 0;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int up = 0; up < 4; ++up)
              for (int xp = 0; xp < 4; ++xp)
                for (int yp = 0; yp < 4; ++yp) {
                  if (!can_pair(m, xp, yp)) continue;
                  int Pin = ptype(yp, xp); /* inner pair seen from the loop: (phi_l, phi_k) */
                  for (int vp = 0; vp < 4; ++vp)
                    for (int tt_ = 0; tt_ < St; ++tt_)
                      A2[((a * 4 + u) * 4 + vp) * St + tt_] +=
                          t->wtm[Pin][vp][up] * A1[((((a * 4 + u) * 4 + up) * 16) + xp * 4 + yp) * St + tt_];
                }
        for (int q = 0; q < Sa * 16 * Sc; ++q) A3[q] = 0;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int vp = 0; vp < 4; ++vp)
              for (int tt_ = 0; tt_ < St; ++tt_) {
                real w = A2[((a * 4 + u) * 4 + vp) * St + tt_];
                if (w == 0) continue;
                for (int v = 0; v < 4; ++v)
                  for (int c = 0; c < Sc; ++c) A3[((a * 4 + u) * 4 + v) * Sc + c] += w * UpR[((tt_ * 4 + vp) * 4 + v) * Sc + c];
              }
        real wi = t->win[l1 + l2];
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            int P = ptype(x, y);
            for (int a = 0; a < Sa; ++a)
              for (int u = 0; u < 4; ++u)
                for (int v = 0; v < 4; ++v)
                  for (int c = 0; c < Sc; ++c)
                    INNER(x, y, a, c) += wi * t->wtm[P][u][v] * A3[((a * 4 + u) * 4 + v) * Sc + c];
          }
      }
    }
  /* multiloop closure: w_a w_c M2(i+1,j-1)[a',c'] */
  if (j - 1 >= i + 1) {
    const real* m2 = t->m2[(size_t)(i + 1) * n + (j - 1)];
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        for (int a = 0; a < Sa; ++a)
          for (int c = 0; c < Sc; ++c) INNER(x, y, a, c) += t->wa * t->wc * m2[a * Sc + c];
      }
  }
  /* dress with T_i, T_j: Qb[a,x,y,c] = can(x,y) sum_{a',c'} T_i[a,x,a'] T_j[c',y,c] inner[x,y;a',c'] */
  const real *Ti = t->Td[i], *Tj = t->Td[j];
  for (int a = 0; a < Si; ++a)
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        for (int c = 0; c < Sj1; ++c) {
          real s = 0;
          for (int ap = 0; ap < Sa; ++ap)
            for (int cp = 0; cp < Sc; ++cp)
              s += Ti[(a * 4 + x) * Sa + ap] * Tj[(cp * 4 + y) * Sj1 + c] * INNER(x, y, ap, cp);
          qb[((a * 4 + x) * 4 + y) * Sj1 + c] = s;
        }
      }
#undef INNER
  free(inner); free(UpL); free(UpR); free(A1); free(A2); free(A3);
}

static void compute_cell(orc_tables* t, int i, int j) {
  int n = t->n;
  int Si = SG(t, i), Sj1 = SG(t, j + 1);
  size_t ci = (size_t)i * n + j;
  compute_qb(t, i, j);
  real *qb = t->qb[ci], *qbs = t->qbs[ci], *qm1 = t->qm1[ci], *qml = t->qml[ci], *m2 = t->m2[ci], *qm = t->qm[ci];
  /* Qbs[a,c] = sum_{x,y} Qb[a,x,y,c] */
  for (int a = 0; a < Si; ++a)
    for (int xy = 0; xy < 16; ++xy)
      for (int c = 0; c < Sj1; ++c) qbs[a * Sj1 + c] += qb[(a * 16 + xy) * Sj1 + c];
  /* Qm1(i,j) = w_c Qbs(i,j) + w_b Qm1(i,j-1) Tbar_j */
  for (int a = 0; a < Si; ++a)
    for (int c = 0; c < Sj1; ++c) qm1[a * Sj1 + c] = t->wc * qbs[a * Sj1 + c];
  if (j - 1 >= i) {
    const real* p = t->qm1[(size_t)i * n + (j - 1)];
    int Sj = SG(t, j);
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Sj; ++s)
        for (int c = 0; c < Sj1; ++c) qm1[a * Sj1 + c] += t->wb * p[a * Sj + s] * t->Tb[j][s * Sj1 + c];
  }
  /* Qml(i,j) = Qm1(i,j) + w_b Tbar_i Qml(i+1,j) */
  for (int k = 0; k < Si * Sj1; ++k) qml[k] = qm1[k];
  if (i + 1 <= j) {
    const real* p = t->qml[(size_t)(i + 1) * n + j];
    int Si1 = SG(t, i + 1);
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Si1; ++s)
        for (int c = 0; c < Sj1; ++c) qml[a * Sj1 + c] += t->wb * t->Tb[i][a * Si1 + s] * p[s * Sj1 + c];
  }
  /* M2(i,j) = sum_{k=i+1}^{j} Qm(i,k-1) Qm1(k,j)   (eq 3.5 first line, line 172, on the packed index space) */
  for (int k = i + 1; k <= j; ++k) {
    const real* A = t->qm[(size_t)i * n + (k - 1)];
    const real* B = t->qm1[(size_t)k * n + j];
    int Sk = SG(t, k);
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Sk; ++s) {
        real w = A[a * Sk + s];
        if (w == 0) continue;
        for (int c = 0; c < Sj1; ++c) m2[a * Sj1 + c] += w * B[s * Sj1 + c];
      }
  }
  for (int k = 0; k < Si * Sj1; ++k) qm[k] = qml[k] + m2[k];
}

static int inside_impl(const orc_model* m, const orc_tt* tt_in, int nthreads, int forbid_i, int forbid_j, orc_tables** out,
                       double* logZ) {
  int n = tt_in->n;
  orc_tables* t = (orc_tables*)calloc(1, sizeof(orc_tables));
  t->n = n;
  t->forbid_i = forbid_i;
  t->forbid_j = forbid_j;
  t->model = *m;
  /* private TT copy */
  t->tt = (orc_tt*)calloc(1, sizeof(orc_tt));
  t->tt->n = n;
  t->tt->sigma = (int*)malloc(sizeof(int) * (n + 1));
  t->tt->start = (int*)malloc(sizeof(int) * (n + 1));
  memcpy(t->tt->sigma, tt_in->sigma, sizeof(int) * (n + 1));
  memcpy(t->tt->start, tt_in->start, sizeof(int) * (n + 1));
  t->tt->ops = (orc_op*)malloc(sizeof(orc_op) * (tt_in->start[n] + 1));
  memcpy(t->tt->ops, tt_in->ops, sizeof(orc_op) * tt_in->start[n]);
  t->sig = t->tt->sigma;
  double kT = model_kT(m);
  t->beta = 1.0 / kT;
  for (int p = 0; p < 6; ++p) {
    for (int q = 0; q < 6; ++q) t->wst[p][q] = expl(-(real)(m->stack[p][q] * t->beta));
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) t->wtm[p][x][y] = expl(-(real)(m->tmm[p][x][y] * t->beta));
  }
  for (int l = 0; l < 31; ++l) {
    t->wbu[l] = l >= 1 ? expl(-(real)(m->bulge_init[l] * t->beta)) : 0;
    t->win[l] = l >= 2 ? expl(-(real)(m->interior_init[l] * t->beta)) : 0;
  }
  t->wa = expl(-(real)(m->ml_a * t->beta));
  t->wb = expl(-(real)(m->ml_b * t->beta));
  t->wc = expl(-(real)(m->ml_c * t->beta));
  /* dense cores (eq S3.7) and transfer matrices */
  t->Td = (real**)calloc(n, sizeof(real*));
  t->Tb = (real**)calloc(n, sizeof(real*));
  for (int i = 0; i < n; ++i) {
    int Sa = SG(t, i), Sc = SG(t, i + 1);
    t->Td[i] = cell_alloc((size_t)Sa * 4 * Sc);
    t->Tb[i] = cell_alloc((size_t)Sa * Sc);
    for (int z = t->tt->start[i]; z < t->tt->start[i + 1]; ++z) {
      const orc_op* o = &t->tt->ops[z];
      t->Td[i][(o->a * 4 + o->b) * Sc + o->c] += (real)o->x;
      t->Tb[i][o->a * Sc + o->c] += (real)o->x;
    }
  }
  /* stretches E(i,j) */
  t->E = (real**)calloc((size_t)(n + 1) * (n + 1), sizeof(real*));
  for (int i = 0; i <= n; ++i) {
    int Sa = SG(t, i);
    real* id = cell_alloc((size_t)Sa * Sa);
    for (int a = 0; a < Sa; ++a) id[a * Sa + a] = 1;
    t->E[(size_t)i * (n + 1) + i] = id; /* E(i,i-1) = I */
    for (int j = i; j < n; ++j) {
      int Sj = SG(t, j), Sj1 = SG(t, j + 1);
      const real* prev = t->E[(size_t)i * (n + 1) + j];
      real* e = cell_alloc((size_t)Sa * Sj1);
      for (int a = 0; a < Sa; ++a)
        for (int s = 0; s < Sj; ++s)
          for (int c = 0; c < Sj1; ++c) e[a * Sj1 + c] += prev[a * Sj + s] * t->Tb[j][s * Sj1 + c];
      t->E[(size_t)i * (n + 1) + (j + 1)] = e;
    }
  }
  size_t nn = (size_t)n * n;
  t->qb = (real**)calloc(nn, sizeof(real*));
  t->qbs = (real**)calloc(nn, sizeof(real*));
  t->qm1 = (real**)calloc(nn, sizeof(real*));
  t->qml = (real**)calloc(nn, sizeof(real*));
  t->m2 = (real**)calloc(nn, sizeof(real*));
  t->qm = (real**)calloc(nn, sizeof(real*));
  for (int i = 0; i < n; ++i)
    for (int j = i; j < n; ++j) {
      size_t ci = (size_t)i * n + j, s2 = (size_t)SG(t, i) * SG(t, j + 1);
      t->qb[ci] = cell_alloc(s2 * 16);
      t->qbs[ci] = cell_alloc(s2);
      t->qm1[ci] = cell_alloc(s2);
      t->qml[ci] = cell_alloc(s2);
      t->m2[ci] = cell_alloc(s2);
      t->qm[ci] = cell_alloc(s2);
    }
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
  for (int d = 0; d < n; ++d) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < n - d; ++i) compute_cell(t, i, i + d);
  }
  /* exterior (eq 3.7): Qext(j) = Qext(j-1) Tbar_j + sum_k Qext(k-1) Qbs(k,j) */
  t->qext = (real**)calloc(n + 1, sizeof(real*));
  t->qext[0] = cell_alloc(SG(t, 0));
  t->qext[0][0] = 1;
  for (int j = 0; j < n; ++j) {
    int Sj = SG(t, j), Sj1 = SG(t, j + 1);
    real* q = cell_alloc(Sj1);
    for (int s = 0; s < Sj; ++s)
      for (int c = 0; c < Sj1; ++c) q[c] += t->qext[j][s] * t->Tb[j][s * Sj1 + c];
    for (int k = 0; k <= j; ++k) {
      const real* qbs = t->qbs[(size_t)k * n + j];
      int Sk = SG(t, k);
      for (int s = 0; s < Sk; ++s)
        for (int c = 0; c < Sj1; ++c) q[c] += t->qext[k][s] * qbs[s * Sj1 + c];
    }
    t->qext[j + 1] = q;
  }
  real Z = 0;
  for (int c = 0; c < SG(t, n); ++c) Z += t->qext[n][c];
  if (logZ) *logZ = (double)logl(Z);
  if (out) *out = t; else orc_tables_free(t);
  return 0;
}

int orc_inside(const orc_model* m, const orc_tt* tt_in, int nthreads, orc_tables** out, double* logZ) {
  return inside_impl(m, tt_in, nthreads, -1, -1, out, logZ);
}

void orc_tables_free(orc_tables* t) {
  if (!t) return;
  int n = t->n;
  for (int i = 0; i < n; ++i) { free(t->Td[i]); free(t->Tb[i]); }
  free(t->Td); free(t->Tb);
  for (size_t k = 0; k < (size_t)(n + 1) * (n + 1); ++k) free(t->E[k]);
  free(t->E);
  for (size_t k = 0; k < (size_t)n * n; ++k) {
    free(t->qb[k]); free(t->qbs[k]); free(t->qm1[k]); free(t->qml[k]); free(t->m2[k]); free(t->qm[k]);
  }
  free(t->qb); free(t->qbs); free(t->qm1); free(t->qml); free(t->m2); free(t->qm);
  for (int j = 0; j <= n; ++j) free(t->qext[j]);
  free(t->qext);
  orc_tt_free(t->tt);
  free(t);
}

int orc_tables_cell(const orc_tables* t, int which, int i, int j, int shift, double* out) {
  if (i < 0 || j < i || j >= t->n) return -1;
  size_t ci = (size_t)i * t->n + j;
  real** tabs[6] = {t->qb, t->qbs, t->qm1, t->qml, t->m2, t->qm};
  if (which < 0 || which > 5) return -1;
  size_t cnt = (size_t)SG(t, i) * SG(t, j + 1) * (which == 0 ? 16 : 1);
  for (size_t k = 0; k < cnt; ++k) out[k] = (double)ldexpl(tabs[which][ci][k], -shift);
  return (int)cnt;
}

double orc_tables_logqext(const orc_tables* t, int j, int c) {
  real v = t->qext[j + 1][c];
  return v > 0 ? (double)logl(v) : -INFINITY;
}

/* ------------------------------------------------------------------------- */
/* stochastic traceback                        */
/* ------------------------------------------------------------------------- */
static uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
double orc_uniform(uint64_t seed, uint64_t sample, uint64_t kind, uint64_t i, uint64_t j) {
  uint64_t h = seed;
  uint64_t v[4] = {sample, kind, i, j};
  for (int k = 0; k < 4; ++k) h = mix64(h + 0x9E3779B97F4A7C15ULL * (v[k] + 1));
  return (double)(h >> 11) * (1.0 / 9007199254740992.0);
}

enum { K_TOP = 0, K_EXT = 1, K_QB = 2, K_QM = 3, K_QML = 4, K_QM1 = 5, K_CHAIN = 6, K_HAIRPIN = 7, K_ILOOP = 8 };
enum { IT_QB = 0, IT_QM = 1, IT_QML = 2, IT_QM1 = 3 };
typedef struct { int type, i, j, a, x, y, c; } tb_item;

/* a growing list of alternative weights; pick() returns the first index whose running sum exceeds u*total */
typedef struct { real* w; int n, cap; } altlist;
static void alt_reset(altlist* L) { L->n = 0; }
static void alt_push(altlist* L, real w) {
  if (L->n == L->cap) { L->cap = L->cap ? 2 * L->cap : 256; L->w = (real*)realloc(L->w, sizeof(real) * L->cap); }
  L->w[L->n++] = w;
}
static int alt_pick(const altlist* L, double u) {
  real tot = 0;
  for (int k = 0; k < L->n; ++k) tot += L->w[k];
  real thr = (real)u * tot, run = 0;
  int last = -1;
  for (int k = 0; k < L->n; ++k) {
    if (L->w[k] <= 0) continue;
    run += L->w[k];
    last = k;
    if (run > thr) return k;
  }
  return last;
}

/* same, with the total taken from the stored table entry that the alternatives decompose */
static int alt_pick_total(const altlist* L, double u, real tot) {
  real thr = (real)u * tot, run = 0;
  int last = -1;
  for (int k = 0; k < L->n; ++k) {
    if (L->w[k] <= 0) continue;
    run += L->w[k];
    last = k;
    if (run > thr) return k;
  }
  return last;
}

typedef struct {
  const orc_tables* t;
  uint64_t seed; int sample;
  uint8_t* seq; int32_t* pair;
  altlist L;
  tb_item* stk; int sp, cap;
} tb_ctx;

static void tb_push(tb_ctx* c, tb_item it) {
  if (c->sp == c->cap) { c->cap = c->cap ? 2 * c->cap : 64; c->stk = (tb_item*)realloc(c->stk, sizeof(tb_item) * c->cap); }
  c->stk[c->sp++] = it;
}
static double tb_u(const tb_ctx* c, int kind, int i, int j) {
  return orc_uniform(c->seed, (uint64_t)c->sample, (uint64_t)kind, (uint64_t)i, (uint64_t)j);
}

/* CHAIN(p,q,s,t): unpaired stretch p..q with fixed end bonds; choose z_m prop. to x(z) b_{m+1}[c(z)],
 * b_m = Tbar_m ... Tbar_q e_t */
static void tb_chain(tb_ctx* c, int p, int q, int s, int tend) {
  const orc_tables* t = c->t;
  if (p > q) return;
  int cur = s;
  for (int mpos = p; mpos <= q; ++mpos) {
    alt_reset(&c->L);
    int z0 = t->tt->start[mpos], z1 = t->tt->start[mpos + 1];
    const real* Er = getE(t, mpos + 1, q); /* b_{m+1}[.] = E(m+1,q)[., tend] */
    int Sq1 = SG(t, q + 1);
    for (int z = z0; z < z1; ++z) {
      const orc_op* o = &t->tt->ops[z];
      alt_push(&c->L, o->a == cur ? (real)o->x * Er[o->c * Sq1 + tend] : 0);
    }
    int k = alt_pick(&c->L, tb_u(c, K_CHAIN, mpos, 0));
    const orc_op* o = &t->tt->ops[z0 + k];
    c->seq[mpos] = (uint8_t)o->b;
    cur = o->c;
  }
}

static void tb_qb(tb_ctx* c, tb_item it) {
  const orc_tables* t = c->t;
  const orc_model* m = &t->model;
  const orc_tt* tt = t->tt;
  int n = t->n, i = it.i, j = it.j, d = j - i, x = it.x, y = it.y;
  int P = ptype(x, y);
  c->seq[i] = (uint8_t)x; c->seq[j] = (uint8_t)y;
  c->pair[i] = j; c->pair[j] = i;
  real wh = expl(-(real)(hairpin_init(m, d - 1) * t->beta));
  int Sc = SG(t, j);
  /* level A, in the order of DESIGN.md "Traceback order":
   *   hairpin | stack | multiloop (k asc, s asc) | one inner pair by l1+l2 = 1,2,.. then l1 asc;
   * within each, the operator pairs (z_i, z_j) in list order (z_i outer).  For the multiloop the
   * operator pair is the outer loop.  The threshold is u * (stored Qb entry). */
  typedef struct { int zi, zj, kind, k, l, s; } altA;
  altA* desc = NULL; int nd = 0, capd = 0;
#define PUSHA(W, ...) do { if (nd == capd) { capd = capd ? 2 * capd : 512; desc = (altA*)realloc(desc, sizeof(altA) * capd); } \
    desc[nd++] = (altA){__VA_ARGS__}; alt_push(&c->L, (W)); } while (0)
  alt_reset(&c->L);
  int maxS = 1;
  for (int p = i; p <= j + 1; ++p) if (SG(t, p) > maxS) maxS = SG(t, p);
  real* UpL = cell_alloc((size_t)maxS * 16 * maxS);
  real* UpR = cell_alloc((size_t)maxS * 16 * maxS);
  /* the operator pairs compatible with (a,x) and (y,c) */
  int npz = 0;
  int* pzi = (int*)calloc((size_t)(tt->start[i + 1] - tt->start[i]) * (tt->start[j + 1] - tt->start[j]) + 1, sizeof(int));
  int* pzj = (int*)calloc((size_t)(tt->start[i + 1] - tt->start[i]) * (tt->start[j + 1] - tt->start[j]) + 1, sizeof(int));
  for (int zi = tt->start[i]; zi < tt->start[i + 1]; ++zi)
    for (int zj = tt->start[j]; zj < tt->start[j + 1]; ++zj) {
      const orc_op *oi = &tt->ops[zi], *oj = &tt->ops[zj];
      if (oi->a != it.a || oi->b != x || oj->b != y || oj->c != it.c) continue;
      pzi[npz] = zi; pzj[npz] = zj; ++npz;
    }
  int tmax = d - 2 - (m->min_hairpin + 1);
  if (tmax > m->max_interior) tmax = m->max_interior;
  for (int seg = 0; seg < 3 + (tmax >= 1 ? tmax : 0); ++seg) {
    /* seg 0 hairpin, 1 stack, 2 multiloop, 3.. one inner pair of total size seg-2 */
    int tot_sz = seg == 1 ? 0 : seg - 2;
    if (seg == 1 && tmax < 0) continue;
    int nl1 = (seg == 0 || seg == 2) ? 1 : tot_sz + 1;
    if (seg == 2) {
      for (int pz = 0; pz < npz; ++pz) {
        const orc_op *oi = &tt->ops[pzi[pz]], *oj = &tt->ops[pzj[pz]];
        real w0 = (real)oi->x * (real)oj->x;
        int ap = oi->c, cp = oj->a;
        for (int k = i + 2; k <= j - 1; ++k) {
          const real* A = t->qm[(size_t)(i + 1) * n + (k - 1)];
          const real* B = t->qm1[(size_t)k * n + (j - 1)];
          int Sk = SG(t, k);
          for (int sb = 0; sb < Sk; ++sb) PUSHA(w0 * t->wa * t->wc * A[ap * Sk + sb] * B[sb * Sc + cp], pzi[pz], pzj[pz], 2, k, 0, sb);
        }
      }
      continue;
    }
    for (int l1 = 0; l1 < nl1; ++l1)
      for (int pz = 0; pz < npz; ++pz) {
        const orc_op *oi = &tt->ops[pzi[pz]], *oj = &tt->ops[pzj[pz]];
        real w0 = (real)oi->x * (real)oj->x;
        int ap = oi->c, cp = oj->a;
        if (seg == 0) {
          compute_Up(t, i + 1, j - 1, UpL);
          real s = 0;
          for (int u = 0; u < 4; ++u)
            for (int v = 0; v < 4; ++v) s += wh * t->wtm[P][u][v] * UpL[((ap * 4 + u) * 4 + v) * Sc + cp];
          PUSHA(w0 * s, pzi[pz], pzj[pz], 0, 0, 0, 0);
          continue;
        }
        int l2 = tot_sz - l1;
        int k = i + 1 + l1, l = j - 1 - l2;
        const real* qin = t->qb[(size_t)k * n + l];
        int Ss = SG(t, k), St = SG(t, l + 1);
        real s = 0;
        for (int xp = 0; xp < 4; ++xp)
          for (int yp = 0; yp < 4; ++yp) {
            if (!can_pair(m, xp, yp)) continue;
            if (l1 == 0 && l2 == 0) {
              s += t->wst[P][ptype(xp, yp)] * qin[((ap * 4 + xp) * 4 + yp) * St + cp];
            } else if (l2 == 0) {
              const real* El = getE(t, i + 1, k - 1);
              real w = t->wbu[l1] * (l1 == 1 ? t->wst[P][ptype(xp, yp)] : 1.0L);
              for (int sb = 0; sb < Ss; ++sb) s += w * El[ap * Ss + sb] * qin[((sb * 4 + xp) * 4 + yp) * St + cp];
            } else if (l1 == 0) {
              const real* Er = getE(t, l + 1, j - 1);
              real w = t->wbu[l2] * (l2 == 1 ? t->wst[P][ptype(xp, yp)] : 1.0L);
              for (int tb = 0; tb < St; ++tb) s += w * qin[((ap * 4 + xp) * 4 + yp) * St + tb] * Er[tb * Sc + cp];
            }
          }
        if (l1 > 0 && l2 > 0) {
          compute_Up(t, i + 1, k - 1, UpL);
          compute_Up(t, l + 1, j - 1, UpR);
          for (int u = 0; u < 4; ++u)
            for (int up = 0; up < 4; ++up)
              for (int sb = 0; sb < Ss; ++sb) {
                real wl = UpL[((ap * 4 + u) * 4 + up) * Ss + sb];
                if (wl == 0) continue;
                for (int xp = 0; xp < 4; ++xp)
                  for (int yp = 0; yp < 4; ++yp) {
                    if (!can_pair(m, xp, yp)) continue;
                    for (int tb = 0; tb < St; ++tb) {
                      real wq = qin[((sb * 4 + xp) * 4 + yp) * St + tb];
                      if (wq == 0) continue;
                      for (int vp = 0; vp < 4; ++vp)
                        for (int v = 0; v < 4; ++v)
                          s += t->win[l1 + l2] * t->wtm[P][u][v] * t->wtm[ptype(yp, xp)][vp][up] * wl * wq *
                               UpR[((tb * 4 + vp) * 4 + v) * Sc + cp];
                    }
                  }
              }
        }
        PUSHA(w0 * s, pzi[pz], pzj[pz], 1, k, l, 0);
      }
  }
  free(pzi); free(pzj);
#undef PUSHA
  int pick = alt_pick_total(&c->L, tb_u(c, K_QB, i, j), t->qb[(size_t)i * n + j][((it.a * 4 + x) * 4 + y) * SG(t, j + 1) + it.c]);
  altA A = desc[pick];
  free(desc);
  const orc_op *oi = &tt->ops[A.zi], *oj = &tt->ops[A.zj];
  int ap = oi->c, cp = oj->a;
  if (A.kind == 0) {
    /* hairpin ends: joint choice of the operators at i+1 and j-1 (K_HAIRPIN), then the interior chain */
    int p = i + 1, q = j - 1;
    const real* Em = getE(t, p + 1, q - 1);
    int Sm = SG(t, q);
    alt_reset(&c->L);
    int zp0 = tt->start[p], zp1 = tt->start[p + 1], zq0 = tt->start[q], zq1 = tt->start[q + 1];
    for (int zp = zp0; zp < zp1; ++zp)
      for (int zq = zq0; zq < zq1; ++zq) {
        const orc_op *o = &tt->ops[zp], *r = &tt->ops[zq];
        real w = 0;
        if (o->a == ap && r->c == cp) w = (real)o->x * (real)r->x * Em[o->c * Sm + r->a] * t->wtm[P][o->b][r->b];
        alt_push(&c->L, w);
      }
    int k = alt_pick(&c->L, tb_u(c, K_HAIRPIN, i, j));
    const orc_op *o = &tt->ops[zp0 + k / (zq1 - zq0)], *r = &tt->ops[zq0 + k % (zq1 - zq0)];
    c->seq[p] = (uint8_t)o->b; c->seq[q] = (uint8_t)r->b;
    tb_chain(c, p + 1, q - 1, o->c, r->a);
  } else if (A.kind == 1) {
    /* one inner pair (k,l): level B (K_ILOOP) chooses the stretch end operators and (x',y') */
    int k = A.k, l = A.l, l1 = k - i - 1, l2 = j - l - 1;
    const real* qin = t->qb[(size_t)k * n + l];
    int St = SG(t, l + 1);
    /* left side alternatives: (operator at i+1, operator at k-1) with resulting (u,u',s) */
    typedef struct { int z1, z2, u, up, s; real w; } side;
    side *Ls = NULL, *Rs = NULL; int nL = 0, nR = 0;
    Ls = (side*)calloc(4096, sizeof(side)); Rs = (side*)calloc(4096, sizeof(side));
    if (l1 == 0) { Ls[nL++] = (side){-1, -1, 0, 0, ap, 1}; }
    else if (l1 == 1) {
      for (int z = tt->start[i + 1]; z < tt->start[i + 2]; ++z) {
        const orc_op* o = &tt->ops[z];
        if (o->a == ap) Ls[nL++] = (side){z, -1, o->b, o->b, o->c, (real)o->x};
      }
    } else {
      const real* Em = getE(t, i + 2, k - 2);
      int Sm = SG(t, k - 1);
      for (int z = tt->start[i + 1]; z < tt->start[i + 2]; ++z)
        for (int z2 = tt->start[k - 1]; z2 < tt->start[k]; ++z2) {
          const orc_op *o = &tt->ops[z], *r = &tt->ops[z2];
          if (o->a == ap) Ls[nL++] = (side){z, z2, o->b, r->b, r->c, (real)o->x * Em[o->c * Sm + r->a] * (real)r->x};
        }
    }
    if (l2 == 0) { Rs[nR++] = (side){-1, -1, 0, 0, cp, 1}; }
    else if (l2 == 1) {
      for (int z = tt->start[j - 1]; z < tt->start[j]; ++z) {
        const orc_op* o = &tt->ops[z];
        if (o->c == cp) Rs[nR++] = (side){z, -1, o->b, o->b, o->a, (real)o->x};
      }
    } else {
      const real* Em = getE(t, l + 2, j - 2);
      int Sm = SG(t, j - 1);
      /* z1 = operator at l+1 (gives v'), z2 = operator at j-1 (gives v); s = left bond of l+1 */
      for (int z = tt->start[l + 1]; z < tt->start[l + 2]; ++z)
        for (int z2 = tt->start[j - 1]; z2 < tt->start[j]; ++z2) {
          const orc_op *o = &tt->ops[z], *r = &tt->ops[z2];
          if (r->c == cp) Rs[nR++] = (side){z, z2, r->b, o->b, o->a, (real)o->x * Em[o->c * Sm + r->a] * (real)r->x};
        }
    }
    /* for the right side: .u = v (at j-1), .up = v' (at l+1), .s = t (right bond of the inner cell) */
    alt_reset(&c->L);
    for (int a_ = 0; a_ < nL; ++a_)
      for (int b_ = 0; b_ < nR; ++b_)
        for (int xp = 0; xp < 4; ++xp)
          for (int yp = 0; yp < 4; ++yp) {
            real w = 0;
            if (can_pair(m, xp, yp)) {
              real e;
              if (l1 == 0 && l2 == 0) e = t->wst[P][ptype(xp, yp)];
              else if (l1 == 0 || l2 == 0) e = t->wbu[l1 + l2] * (l1 + l2 == 1 ? t->wst[P][ptype(xp, yp)] : 1.0L);
              else e = t->win[l1 + l2] * t->wtm[P][Ls[a_].u][Rs[b_].u] * t->wtm[ptype(yp, xp)][Rs[b_].up][Ls[a_].up];
              w = e * Ls[a_].w * Rs[b_].w * qin[((Ls[a_].s * 4 + xp) * 4 + yp) * St + Rs[b_].s];
            }
            alt_push(&c->L, w);
          }
    int pk = alt_pick(&c->L, tb_u(c, K_ILOOP, i, j));
    int yp = pk % 4, xp = (pk / 4) % 4, b_ = (pk / 16) % nR, a_ = pk / (16 * nR);
    side SL = Ls[a_], SR = Rs[b_];
    if (l1 == 1) { c->seq[i + 1] = (uint8_t)SL.u; }
    else if (l1 >= 2) {
      c->seq[i + 1] = (uint8_t)SL.u; c->seq[k - 1] = (uint8_t)SL.up;
      tb_chain(c, i + 2, k - 2, tt->ops[SL.z1].c, tt->ops[SL.z2].a);
    }
    if (l2 == 1) { c->seq[j - 1] = (uint8_t)SR.u; }
    else if (l2 >= 2) {
      c->seq[j - 1] = (uint8_t)SR.u; c->seq[l + 1] = (uint8_t)SR.up;
      tb_chain(c, l + 2, j - 2, tt->ops[SR.z1].c, tt->ops[SR.z2].a);
    }
    tb_push(c, (tb_item){IT_QB, k, l, SL.s, xp, yp, SR.s});
    free(Ls); free(Rs);
  } else {
    tb_push(c, (tb_item){IT_QM, i + 1, A.k - 1, ap, 0, 0, A.s});
    tb_push(c, (tb_item){IT_QM1, A.k, j - 1, A.s, 0, 0, cp});
  }
  free(UpL); free(UpR);
}

static void tb_run(tb_ctx* c) {
  const orc_tables* t = c->t;
  const orc_model* m = &t->model;
  const orc_tt* tt = t->tt;
  int n = t->n;
  for (int p = 0; p < n; ++p) { c->seq[p] = 255; c->pair[p] = -1; }
  c->sp = 0;
  /* TOP */
  alt_reset(&c->L);
  for (int cc = 0; cc < SG(t, n); ++cc) alt_push(&c->L, t->qext[n][cc]);
  int cb = alt_pick(&c->L, tb_u(c, K_TOP, 0, 0));
  /* EXT(j,c) */
  int j = n - 1;
  while (j >= 0) {
    alt_reset(&c->L);
    int z0 = tt->start[j], z1 = tt->start[j + 1];
    for (int z = z0; z < z1; ++z) {
      const orc_op* o = &tt->ops[z];
      alt_push(&c->L, o->c == cb ? t->qext[j][o->a] * (real)o->x : 0);
    }
    int nops = z1 - z0;
    int Sj1 = SG(t, j + 1);
    /* k ascending, s ascending, (x,y) lexicographic */
    int* koff = (int*)calloc(j + 2, sizeof(int));
    for (int k = 0; k <= j - (m->min_hairpin + 1); ++k) {
      koff[k] = c->L.n;
      const real* qb = t->qb[(size_t)k * n + j];
      for (int s = 0; s < SG(t, k); ++s)
        for (int xy = 0; xy < 16; ++xy) alt_push(&c->L, t->qext[k][s] * qb[(s * 16 + xy) * Sj1 + cb]);
    }
    int pk = alt_pick_total(&c->L, tb_u(c, K_EXT, j, 0), t->qext[j + 1][cb]);
    if (pk < nops) {
      const orc_op* o = &tt->ops[z0 + pk];
      c->seq[j] = (uint8_t)o->b;
      cb = o->a;
      j = j - 1;
    } else {
      int k = 0;
      while (k + 1 <= j - (m->min_hairpin + 1) && koff[k + 1] <= pk) ++k;
      int r = pk - koff[k];
      int s = r / 16, xy = r % 16;
      tb_push(c, (tb_item){IT_QB, k, j, s, xy / 4, xy % 4, cb});
      cb = s;
      j = k - 1;
    }
    free(koff);
  }
  while (c->sp > 0) {
    tb_item it = c->stk[--c->sp];
    int i = it.i;
    j = it.j;
    int Sj1 = SG(t, j + 1);
    if (it.type == IT_QB) {
      tb_qb(c, it);
    } else if (it.type == IT_QM) {
      /* QM(i,j,a,c): {QML part}, then {k asc, s asc: Qm(i,k-1)[a,s] Qm1(k,j)[s,c]} */
      alt_reset(&c->L);
      alt_push(&c->L, t->qml[(size_t)i * n + j][it.a * Sj1 + it.c]);
      int* koff = (int*)calloc(j + 2, sizeof(int));
      for (int k = i + 1; k <= j; ++k) {
        koff[k] = c->L.n;
        const real* A = t->qm[(size_t)i * n + (k - 1)];
        const real* B = t->qm1[(size_t)k * n + j];
        int Sk = SG(t, k);
        for (int s = 0; s < Sk; ++s) alt_push(&c->L, A[it.a * Sk + s] * B[s * Sj1 + it.c]);
      }
      int pk = alt_pick_total(&c->L, tb_u(c, K_QM, i, j), t->qm[(size_t)i * n + j][it.a * Sj1 + it.c]);
      if (pk == 0) tb_push(c, (tb_item){IT_QML, i, j, it.a, 0, 0, it.c});
      else {
        int k = i + 1;
        while (k + 1 <= j && koff[k + 1] <= pk) ++k;
        int s = pk - koff[k];
        tb_push(c, (tb_item){IT_QM, i, k - 1, it.a, 0, 0, s});
        tb_push(c, (tb_item){IT_QM1, k, j, s, 0, 0, it.c});
      }
      free(koff);
    } else if (it.type == IT_QML) {
      /* QML(i,j,a,c): {Qm1(i,j)[a,c]}, then {z at i with a(z)=a: w_b x(z) Qml(i+1,j)[c(z),c]} */
      alt_reset(&c->L);
      alt_push(&c->L, t->qm1[(size_t)i * n + j][it.a * Sj1 + it.c]);
      int z0 = tt->start[i], z1 = tt->start[i + 1];
      for (int z = z0; z < z1; ++z) {
        const orc_op* o = &tt->ops[z];
        real w = 0;
        if (o->a == it.a && i + 1 <= j) w = t->wb * (real)o->x * t->qml[(size_t)(i + 1) * n + j][o->c * Sj1 + it.c];
        alt_push(&c->L, w);
      }
      int pk = alt_pick_total(&c->L, tb_u(c, K_QML, i, j), t->qml[(size_t)i * n + j][it.a * Sj1 + it.c]);
      if (pk == 0) tb_push(c, (tb_item){IT_QM1, i, j, it.a, 0, 0, it.c});
      else {
        const orc_op* o = &tt->ops[z0 + pk - 1];
        c->seq[i] = (uint8_t)o->b;
        tb_push(c, (tb_item){IT_QML, i + 1, j, o->c, 0, 0, it.c});
      }
    } else {
      /* QM1(i,j,a,c): {(x,y): w_c Qb(i,j)[a,x,y,c]}, then {z at j with c(z)=c: w_b Qm1(i,j-1)[a,a(z)] x(z)} */
      alt_reset(&c->L);
      const real* qb = t->qb[(size_t)i * n + j];
      for (int xy = 0; xy < 16; ++xy) alt_push(&c->L, t->wc * qb[(it.a * 16 + xy) * Sj1 + it.c]);
      int z0 = tt->start[j], z1 = tt->start[j + 1];
      for (int z = z0; z < z1; ++z) {
        const orc_op* o = &tt->ops[z];
        real w = 0;
        if (o->c == it.c && j - 1 >= i) w = t->wb * t->qm1[(size_t)i * n + (j - 1)][it.a * SG(t, j) + o->a] * (real)o->x;
        alt_push(&c->L, w);
      }
      int pk = alt_pick_total(&c->L, tb_u(c, K_QM1, i, j), t->qm1[(size_t)i * n + j][it.a * Sj1 + it.c]);
      if (pk < 16) tb_push(c, (tb_item){IT_QB, i, j, it.a, pk / 4, pk % 4, it.c});
      else {
        const orc_op* o = &tt->ops[z0 + pk - 16];
        c->seq[j] = (uint8_t)o->b;
        tb_push(c, (tb_item){IT_QM1, i, j - 1, it.a, 0, 0, o->a});
      }
    }
  }
}

int orc_sample(const orc_tables* t, int J, uint64_t seed, uint8_t* seq, int32_t* pair) {
  int n = t->n;
#pragma omp parallel
  {
    tb_ctx c;
    memset(&c, 0, sizeof(c));
    c.t = t; c.seed = seed;
#pragma omp for schedule(dynamic, 1)
    for (int s = 0; s < J; ++s) {
      c.sample = s;
      c.seq = seq + (size_t)s * n;
      c.pair = pair + (size_t)s * n;
      tb_run(&c);
    }
    free(c.L.w); free(c.stk);
  }
  return 0;
}

/* Marginals by their definitions as constrained sums (eqs 2.5-2.7, lines 85-96), each ratio taken from a full inside
 * pass over a restricted ensemble -- O(n^2) passes, for small designs only (the fast way is an outside pass; this is the
 * definition written out):
 *   P(i.j)        = 1 - Z[pair (i,j) forbidden] / Z      (a structure either contains the pair or it does not)
 *   P(phi_m = b)  = Z[operators at m restricted to nucleotide b] / Z
 *   p_k(codon)    = Z[operators at 3k, 3k+1, 3k+2 restricted to the codon's three nucleotides] / Z
 * bpp: upper triangle P(i.j), diagonal P(i unpaired) = 1 - sum_j P(i.j). */
static double restricted_logz(const orc_tables* t, int npos, const int* pos, const int* nuc) {
  const orc_tt* src = t->tt;
  int n = src->n;
  orc_tt r;
  r.n = n;
  r.sigma = src->sigma;
  r.start = (int*)malloc(sizeof(int) * (n + 1));
  r.ops = (orc_op*)malloc(sizeof(orc_op) * (src->start[n] + 1));
  int k = 0, empty = 0;
  for (int i = 0; i < n; ++i) {
    r.start[i] = k;
    int want = -1;
    for (int q = 0; q < npos; ++q)
      if (pos[q] == i) want = nuc[q];
    for (int z = src->start[i]; z < src->start[i + 1]; ++z)
      if (want < 0 || src->ops[z].b == want) r.ops[k++] = src->ops[z];
    if (k == r.start[i]) empty = 1;
  }
  r.start[n] = k;
  double lz = -INFINITY;
  if (!empty) inside_impl(&t->model, &r, 0, -1, -1, NULL, &lz);
  free(r.start);
  free(r.ops);
  return lz;
}

int orc_marginals(orc_tables* t, double* bpp, double* base, double* codon) {
  int n = t->n;
  real Z = 0;
  for (int c = 0; c < SG(t, n); ++c) Z += t->qext[n][c];
  double logZ = (double)logl(Z);
  if (bpp) {
    for (int k = 0; k < n * n; ++k) bpp[k] = 0;
    for (int i = 0; i < n; ++i)
      for (int j = i + t->model.min_hairpin + 1; j < n; ++j) {
        double lz = 0;
        inside_impl(&t->model, t->tt, 0, i, j, NULL, &lz);
        double p = -expm1(lz - logZ);
        bpp[i * n + j] = p > 0 ? p : 0;
      }
    for (int i = 0; i < n; ++i) {
      double s = 0;
      for (int j = 0; j < n; ++j) s += j > i ? bpp[i * n + j] : (j < i ? bpp[j * n + i] : 0);
      bpp[i * n + i] = 1.0 - s;
    }
  }
  if (base)
    for (int m = 0; m < n; ++m)
      for (int b = 0; b < 4; ++b) base[m * 4 + b] = exp(restricted_logz(t, 1, &m, &b) - logZ);
  if (codon)
    for (int k = 0; k < n / 3; ++k)
      for (int c = 0; c < 64; ++c) {
        int pos[3] = {3 * k, 3 * k + 1, 3 * k + 2}, nuc[3] = {c >> 4, (c >> 2) & 3, c & 3};
        codon[k * 64 + c] = exp(restricted_logz(t, 3, pos, nuc) - logZ);
      }
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Minimisation, eq 2.8 (line 102), S4d (lines 245-260), Alg S4.5     */
/* (lines 706-749): the same recursion with every (+, x) of the SumProduct     */
/* semiring replaced by (min, +) of the tropical semiring.                     */
/*   f(z, s) = E(phi(z), s)/kT + sum_i -log x(z_i)    over operator paths z    */
/*   (one operator per position, bonds matching) and structures s;             */
/*   f_min = min f,  one minimiser returned.                                   */
/* "The soft constraint bonus is returned as a free energy ... by taking the   */
/* negative logarithm" (line 749).  Values in units of kT: f_min >= -log Z.    */
/* ------------------------------------------------------------------------- */
#define FINF (1.0e300L)
typedef struct {
  int n;
  const orc_tt* tt;
  const orc_model* m;
  int* sig;
  double beta;
  real** Tc;  /* Tc[i][(a*4+x)*sig[i+1]+c] = min over operators (a,x,c) of -log x   */
  real** Tm;  /* Tm[i][a*sig[i+1]+c]       = min over x                              */
  real** E;   /* min-plus stretch products, index i*(n+1)+(j+1)                      */
  real **fb, **fbs, **fm1, **fml, **fm2, **fm, **fext;
} mfe_tab;

static real rmin(real a, real b) { return a < b ? a : b; }
static real* inf_alloc(size_t k) {
  real* p = (real*)malloc(sizeof(real) * (k ? k : 1));
  for (size_t q = 0; q < (k ? k : 1); ++q) p[q] = FINF;
  return p;
}
static const real* mfeE(const mfe_tab* t, int i, int j) { return t->E[(size_t)i * (t->n + 1) + (j + 1)]; }

/* Up(p,q)[a,u,v,c] = min T_p[a,u,.] + E(p+1,q-1) + T_q[.,v,c]  (p<q);  Up(p,p)[a,u,u,c] = T_p[a,u,c] */
static void mfe_Up(const mfe_tab* t, int p, int q, real* out) {
  int Sa = t->sig[p], Sc = t->sig[q + 1];
  for (int k = 0; k < Sa * 16 * Sc; ++k) out[k] = FINF;
  const orc_tt* tt = t->tt;
  if (p == q) {
    for (int z = tt->start[p]; z < tt->start[p + 1]; ++z) {
      const orc_op* o = &tt->ops[z];
      real* e = &out[((o->a * 4 + o->b) * 4 + o->b) * Sc + o->c];
      *e = rmin(*e, -logl((real)o->x));
    }
    return;
  }
  const real* Em = mfeE(t, p + 1, q - 1);
  int Sm = t->sig[q];
  for (int z = tt->start[p]; z < tt->start[p + 1]; ++z)
    for (int y = tt->start[q]; y < tt->start[q + 1]; ++y) {
      const orc_op *o = &tt->ops[z], *r = &tt->ops[y];
      real* e = &out[((o->a * 4 + o->b) * 4 + r->b) * Sc + r->c];
      *e = rmin(*e, -logl((real)o->x) + Em[o->c * Sm + r->a] - logl((real)r->x));
    }
}

/* one closed cell in the tropical semiring: SURVEY App. A.2 term by term, (+, x) -> (min, +) */
static void mfe_fb(mfe_tab* t, int i, int j) {
  const orc_model* m = t->m;
  int n = t->n, d = j - i;
  int Si = t->sig[i], Sj1 = t->sig[j + 1];
  real* fb = t->fb[(size_t)i * n + j];
  if (d < m->min_hairpin + 1) return;
  real B = (real)t->beta;
  int Sa = t->sig[i + 1], Sc = t->sig[j];
  real* inner = inf_alloc((size_t)16 * Sa * Sc);
#define INNER(x, y, a, c) inner[(((x) * 4 + (y)) * Sa + (a)) * Sc + (c)]
  int maxS = 1;
  for (int p = i; p <= j + 1; ++p) if (t->sig[p] > maxS) maxS = t->sig[p];
  real* UpL = inf_alloc((size_t)maxS * 16 * maxS);
  real* UpR = inf_alloc((size_t)maxS * 16 * maxS);
  real* A1 = inf_alloc((size_t)maxS * 16 * 16 * maxS);
  real* A2 = inf_alloc((size_t)maxS * 16 * maxS);
  real* A3 = inf_alloc((size_t)maxS * 16 * maxS);
  /* hairpin */
  {
    mfe_Up(t, i + 1, j - 1, UpL);
    real gh = B * (real)hairpin_init(m, d - 1);
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        int P = ptype(x, y);
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int v = 0; v < 4; ++v)
              for (int c = 0; c < Sc; ++c)
                INNER(x, y, a, c) = rmin(INNER(x, y, a, c), gh + B * (real)m->tmm[P][u][v] + UpL[((a * 4 + u) * 4 + v) * Sc + c]);
      }
  }
  for (int k = i + 1; k < j; ++k)
    for (int l = j - 1; l > k; --l) {
      int l1 = k - i - 1, l2 = j - l - 1;
      if (l1 + l2 > m->max_interior) break;
      if (l - k < m->min_hairpin + 1) continue;
      const real* qin = t->fb[(size_t)k * n + l];
      int Ss = t->sig[k], St = t->sig[l + 1];
      if (l1 == 0 || l2 == 0) {
        /* stack / bulges: weight by size (+ stack term for sizes 0 and 1), side stretch = min-plus E */
        const real* El = l1 > 0 ? mfeE(t, i + 1, k - 1) : NULL;
        const real* Er = l2 > 0 ? mfeE(t, l + 1, j - 1) : NULL;
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            for (int xp = 0; xp < 4; ++xp)
              for (int yp = 0; yp < 4; ++yp) {
                if (!can_pair(m, xp, yp)) continue;
                real w = (l1 + l2 == 0) ? B * (real)m->stack[ptype(x, y)][ptype(xp, yp)]
                                        : B * (real)(m->bulge_init[l1 + l2] + (l1 + l2 == 1 ? m->stack[ptype(x, y)][ptype(xp, yp)] : 0.0));
                for (int a = 0; a < Sa; ++a)
                  for (int c = 0; c < Sc; ++c) {
                    real best = FINF;
                    if (l1 == 0 && l2 == 0) best = qin[((a * 4 + xp) * 4 + yp) * St + c];
                    else if (l2 == 0) { for (int s = 0; s < Ss; ++s) best = rmin(best, El[a * Ss + s] + qin[((s * 4 + xp) * 4 + yp) * St + c]); }
                    else { for (int tt_ = 0; tt_ < St; ++tt_) best = rmin(best, qin[((a * 4 + xp) * 4 + yp) * St + tt_] + Er[tt_ * Sc + c]); }
                    INNER(x, y, a, c) = rmin(INNER(x, y, a, c), w + best);
                  }
              }
          }
      } else {
        /* generic interior loop, the four stages of compute_qb in (min, +) */
        mfe_Up(t, i + 1, k - 1, UpL);
        mfe_Up(t, l + 1, j - 1, UpR);
        for (int q = 0; q < Sa * 16 * 16 * St; ++q) A1[q] = FINF;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int up = 0; up < 4; ++up)
              for (int s = 0; s < Ss; ++s) {
                real w = UpL[((a * 4 + u) * 4 + up) * Ss + s];
                if (w >= FINF) continue;
                for (int xy = 0; xy < 16; ++xy)
                  for (int tt_ = 0; tt_ < St; ++tt_) {
                    real* e = &A1[((((a * 4 + u) * 4 + up) * 16) + xy) * St + tt_];
                    *e = rmin(*e, w + qin[(s * 16 + xy) * St + tt_]);
                  }
              }
        for (int q = 0; q < Sa * 16 * St; ++q) A2[q] = FINF;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int up = 0; up < 4; ++up)
              for (int xp = 0; xp < 4; ++xp)
                for (int yp = 0; yp < 4; ++yp) {
                  if (!can_pair(m, xp, yp)) continue;
                  int Pin = ptype(yp, xp);
                  for (int vp = 0; vp < 4; ++vp)
                    for (int tt_ = 0; tt_ < St; ++tt_) {
                      real* e = &A2[((a * 4 + u) * 4 + vp) * St + tt_];
                      *e = rmin(*e, B * (real)m->tmm[Pin][vp][up] + A1[((((a * 4 + u) * 4 + up) * 16) + xp * 4 + yp) * St + tt_]);
                    }
                }
        for (int q = 0; q < Sa * 16 * Sc; ++q) A3[q] = FINF;
        for (int a = 0; a < Sa; ++a)
          for (int u = 0; u < 4; ++u)
            for (int vp = 0; vp < 4; ++vp)
              for (int tt_ = 0; tt_ < St; ++tt_) {
                real w = A2[((a * 4 + u) * 4 + vp) * St + tt_];
                if (w >= FINF) continue;
                for (int v = 0; v < 4; ++v)
                  for (int c = 0; c < Sc; ++c) {
                    real* e = &A3[((a * 4 + u) * 4 + v) * Sc + c];
                    *e = rmin(*e, w + UpR[((tt_ * 4 + vp) * 4 + v) * Sc + c]);
                  }
              }
        real gi = B * (real)m->interior_init[l1 + l2];
        for (int x = 0; x < 4; ++x)
          for (int y = 0; y < 4; ++y) {
            if (!can_pair(m, x, y)) continue;
            int P = ptype(x, y);
            for (int a = 0; a < Sa; ++a)
              for (int u = 0; u < 4; ++u)
                for (int v = 0; v < 4; ++v)
                  for (int c = 0; c < Sc; ++c)
                    INNER(x, y, a, c) = rmin(INNER(x, y, a, c), gi + B * (real)m->tmm[P][u][v] + A3[((a * 4 + u) * 4 + v) * Sc + c]);
          }
      }
    }
  /* multiloop closure */
  if (j - 1 >= i + 1) {
    const real* m2 = t->fm2[(size_t)(i + 1) * n + (j - 1)];
    real gac = B * (real)(m->ml_a + m->ml_c);
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        for (int a = 0; a < Sa; ++a)
          for (int c = 0; c < Sc; ++c) INNER(x, y, a, c) = rmin(INNER(x, y, a, c), gac + m2[a * Sc + c]);
      }
  }
  const real *Ti = t->Tc[i], *Tj = t->Tc[j];
  for (int a = 0; a < Si; ++a)
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) {
        if (!can_pair(m, x, y)) continue;
        for (int c = 0; c < Sj1; ++c) {
          real s = FINF;
          for (int ap = 0; ap < Sa; ++ap)
            for (int cp = 0; cp < Sc; ++cp) s = rmin(s, Ti[(a * 4 + x) * Sa + ap] + Tj[(cp * 4 + y) * Sj1 + c] + INNER(x, y, ap, cp));
          fb[((a * 4 + x) * 4 + y) * Sj1 + c] = s;
        }
      }
#undef INNER
  free(inner); free(UpL); free(UpR); free(A1); free(A2); free(A3);
}

static void mfe_cell(mfe_tab* t, int i, int j) {
  const orc_model* m = t->m;
  int n = t->n, Si = t->sig[i], Sj1 = t->sig[j + 1];
  size_t ci = (size_t)i * n + j;
  real B = (real)t->beta, gb = B * (real)m->ml_b, gc = B * (real)m->ml_c;
  mfe_fb(t, i, j);
  real *fb = t->fb[ci], *fbs = t->fbs[ci], *fm1 = t->fm1[ci], *fml = t->fml[ci], *fm2 = t->fm2[ci], *fm = t->fm[ci];
  for (int a = 0; a < Si; ++a)
    for (int xy = 0; xy < 16; ++xy)
      for (int c = 0; c < Sj1; ++c) fbs[a * Sj1 + c] = rmin(fbs[a * Sj1 + c], fb[(a * 16 + xy) * Sj1 + c]);
  for (int k = 0; k < Si * Sj1; ++k) fm1[k] = gc + fbs[k];
  if (j - 1 >= i) {
    const real* p = t->fm1[(size_t)i * n + (j - 1)];
    int Sj = t->sig[j];
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Sj; ++s)
        for (int c = 0; c < Sj1; ++c) fm1[a * Sj1 + c] = rmin(fm1[a * Sj1 + c], gb + p[a * Sj + s] + t->Tm[j][s * Sj1 + c]);
  }
  for (int k = 0; k < Si * Sj1; ++k) fml[k] = fm1[k];
  if (i + 1 <= j) {
    const real* p = t->fml[(size_t)(i + 1) * n + j];
    int Si1 = t->sig[i + 1];
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Si1; ++s)
        for (int c = 0; c < Sj1; ++c) fml[a * Sj1 + c] = rmin(fml[a * Sj1 + c], gb + t->Tm[i][a * Si1 + s] + p[s * Sj1 + c]);
  }
  for (int k = i + 1; k <= j; ++k) {
    const real* A = t->fm[(size_t)i * n + (k - 1)];
    const real* Bq = t->fm1[(size_t)k * n + j];
    int Sk = t->sig[k];
    for (int a = 0; a < Si; ++a)
      for (int s = 0; s < Sk; ++s)
        for (int c = 0; c < Sj1; ++c) fm2[a * Sj1 + c] = rmin(fm2[a * Sj1 + c], A[a * Sk + s] + Bq[s * Sj1 + c]);
  }
  for (int k = 0; k < Si * Sj1; ++k) fm[k] = rmin(fml[k], fm2[k]);
}

static mfe_tab* mfe_build(const orc_model* m, const orc_tt* tt) {
  int n = tt->n;
  mfe_tab* t = (mfe_tab*)calloc(1, sizeof(mfe_tab));
  t->n = n; t->tt = tt; t->m = m; t->sig = tt->sigma;
  t->beta = 1.0 / model_kT(m);
  t->Tc = (real**)calloc(n, sizeof(real*));
  t->Tm = (real**)calloc(n, sizeof(real*));
  for (int i = 0; i < n; ++i) {
    int Sa = t->sig[i], Sc = t->sig[i + 1];
    t->Tc[i] = inf_alloc((size_t)Sa * 4 * Sc);
    t->Tm[i] = inf_alloc((size_t)Sa * Sc);
    for (int z = tt->start[i]; z < tt->start[i + 1]; ++z) {
      const orc_op* o = &tt->ops[z];
      real c = -logl((real)o->x);
      real* e = &t->Tc[i][(o->a * 4 + o->b) * Sc + o->c];
      *e = rmin(*e, c);
      e = &t->Tm[i][o->a * Sc + o->c];
      *e = rmin(*e, c);
    }
  }
  t->E = (real**)calloc((size_t)(n + 1) * (n + 1), sizeof(real*));
  for (int i = 0; i <= n; ++i) {
    int Sa = t->sig[i];
    real* id = inf_alloc((size_t)Sa * Sa);
    for (int a = 0; a < Sa; ++a) id[a * Sa + a] = 0;
    t->E[(size_t)i * (n + 1) + i] = id;
    for (int j = i; j < n; ++j) {
      int Sj = t->sig[j], Sj1 = t->sig[j + 1];
      const real* prev = t->E[(size_t)i * (n + 1) + j];
      real* e = inf_alloc((size_t)Sa * Sj1);
      for (int a = 0; a < Sa; ++a)
        for (int s = 0; s < Sj; ++s)
          for (int c = 0; c < Sj1; ++c) e[a * Sj1 + c] = rmin(e[a * Sj1 + c], prev[a * Sj + s] + t->Tm[j][s * Sj1 + c]);
      t->E[(size_t)i * (n + 1) + (j + 1)] = e;
    }
  }
  size_t nn = (size_t)n * n;
  real*** tabs[6] = {&t->fb, &t->fbs, &t->fm1, &t->fml, &t->fm2, &t->fm};
  for (int w = 0; w < 6; ++w) *tabs[w] = (real**)calloc(nn, sizeof(real*));
  for (int i = 0; i < n; ++i)
    for (int j = i; j < n; ++j) {
      size_t ci = (size_t)i * n + j, s2 = (size_t)t->sig[i] * t->sig[j + 1];
      t->fb[ci] = inf_alloc(s2 * 16);
      for (int w = 1; w < 6; ++w) (*tabs[w])[ci] = inf_alloc(s2);
    }
  for (int d = 0; d < n; ++d) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < n - d; ++i) mfe_cell(t, i, i + d);
  }
  t->fext = (real**)calloc(n + 1, sizeof(real*));
  t->fext[0] = inf_alloc(t->sig[0]);
  t->fext[0][0] = 0;
  for (int j = 0; j < n; ++j) {
    int Sj = t->sig[j], Sj1 = t->sig[j + 1];
    real* q = inf_alloc(Sj1);
    for (int s = 0; s < Sj; ++s)
      for (int c = 0; c < Sj1; ++c) q[c] = rmin(q[c], t->fext[j][s] + t->Tm[j][s * Sj1 + c]);
    for (int k = 0; k <= j; ++k) {
      const real* fbs = t->fbs[(size_t)k * n + j];
      int Sk = t->sig[k];
      for (int s = 0; s < Sk; ++s)
        for (int c = 0; c < Sj1; ++c) q[c] = rmin(q[c], t->fext[k][s] + fbs[s * Sj1 + c]);
    }
    t->fext[j + 1] = q;
  }
  return t;
}

static void mfe_free(mfe_tab* t) {
  int n = t->n;
  for (int i = 0; i < n; ++i) { free(t->Tc[i]); free(t->Tm[i]); }
  free(t->Tc); free(t->Tm);
  for (size_t k = 0; k < (size_t)(n + 1) * (n + 1); ++k) free(t->E[k]);
  free(t->E);
  for (size_t k = 0; k < (size_t)n * n; ++k) { free(t->fb[k]); free(t->fbs[k]); free(t->fm1[k]); free(t->fml[k]); free(t->fm2[k]); free(t->fm[k]); }
  free(t->fb); free(t->fbs); free(t->fm1); free(t->fml); free(t->fm2); free(t->fm);
  for (int j = 0; j <= n; ++j) free(t->fext[j]);
  free(t->fext);
  free(t);
}

/* ---- argmin traceback: every decision recomputes its alternatives in the plain form and follows the smallest ------------------ */
typedef struct { const mfe_tab* t; uint8_t* seq; int32_t* pair; } mfe_tb;
static real opcost(const orc_op* o) { return -logl((real)o->x); }

/* unpaired stretch p..q with end bonds (s, tend): operator by operator, smallest remaining cost */
static void mfe_chain(mfe_tb* c, int p, int q, int s, int tend) {
  const mfe_tab* t = c->t;
  int cur = s;
  for (int mp = p; mp <= q; ++mp) {
    const real* Er = mfeE(t, mp + 1, q);
    int Sq1 = t->sig[q + 1], best = -1;
    real bv = FINF;
    for (int z = t->tt->start[mp]; z < t->tt->start[mp + 1]; ++z) {
      const orc_op* o = &t->tt->ops[z];
      if (o->a != cur) continue;
      real v = opcost(o) + Er[o->c * Sq1 + tend];
      if (v < bv) { bv = v; best = z; }
    }
    c->seq[mp] = (uint8_t)t->tt->ops[best].b;
    cur = t->tt->ops[best].c;
  }
}

static void mfe_tb_fm(mfe_tb* c, int i, int j, int a, int cc);
static void mfe_tb_fm1(mfe_tb* c, int i, int j, int a, int cc);

static void mfe_tb_fb(mfe_tb* c, int i, int j, int a, int x, int y, int cc) {
  const mfe_tab* t = c->t;
  const orc_model* m = t->m;
  const orc_tt* tt = t->tt;
  int n = t->n, d = j - i, P = ptype(x, y);
  real B = (real)t->beta;
  c->seq[i] = (uint8_t)x; c->seq[j] = (uint8_t)y;
  c->pair[i] = j; c->pair[j] = i;
  /* best alternative: kind 0 hairpin (zp,zq) | 1 inner pair (k,l) with side operators | 2 multiloop (k,s) */
  real bv = FINF;
  int bk = -1, bzi = -1, bzj = -1, b1 = -1, b2 = -1, b3 = -1, b4 = -1, bkk = 0, bll = 0, bxp = 0, byp = 0, bs = 0, bt = 0;
  for (int zi = tt->start[i]; zi < tt->start[i + 1]; ++zi)
    for (int zj = tt->start[j]; zj < tt->start[j + 1]; ++zj) {
      const orc_op *oi = &tt->ops[zi], *oj = &tt->ops[zj];
      if (oi->a != a || oi->b != x || oj->b != y || oj->c != cc) continue;
      real w0 = opcost(oi) + opcost(oj);
      int ap = oi->c, cp = oj->a, p = i + 1, q = j - 1;
      /* hairpin */
      {
        const real* Em = mfeE(t, p + 1, q - 1);
        int Sm = t->sig[q];
        real gh = B * (real)hairpin_init(m, d - 1);
        for (int zp = tt->start[p]; zp < tt->start[p + 1]; ++zp)
          for (int zq = tt->start[q]; zq < tt->start[q + 1]; ++zq) {
            const orc_op *o = &tt->ops[zp], *r = &tt->ops[zq];
            if (o->a != ap || r->c != cp) continue;
            real v = w0 + gh + B * (real)m->tmm[P][o->b][r->b] + opcost(o) + Em[o->c * Sm + r->a] + opcost(r);
            if (v < bv) { bv = v; bk = 0; bzi = zi; bzj = zj; b1 = zp; b2 = zq; }
          }
      }
      /* one inner pair */
      for (int k = i + 1; k < j; ++k)
        for (int l = j - 1; l > k; --l) {
          int l1 = k - i - 1, l2 = j - l - 1;
          if (l1 + l2 > m->max_interior) break;
          if (l - k < m->min_hairpin + 1) continue;
          const real* qin = t->fb[(size_t)k * n + l];
          int St = t->sig[l + 1];
          /* left side: (z1 at i+1, z2 at k-1) -> (u, u', s, cost); right side: (z1' at l+1, z2' at j-1) -> (v', v, t, cost) */
          int nl = l1 == 0 ? 1 : (l1 == 1 ? tt->start[i + 2] - tt->start[i + 1] : (tt->start[i + 2] - tt->start[i + 1]) * (tt->start[k] - tt->start[k - 1]));
          int nr = l2 == 0 ? 1 : (l2 == 1 ? tt->start[j] - tt->start[j - 1] : (tt->start[l + 2] - tt->start[l + 1]) * (tt->start[j] - tt->start[j - 1]));
          for (int la = 0; la < nl; ++la) {
            int z1 = -1, z2 = -1, u = 0, up = 0, s = ap;
            real wl = 0;
            if (l1 == 1) {
              z1 = tt->start[i + 1] + la;
              const orc_op* o = &tt->ops[z1];
              if (o->a != ap) continue;
              u = up = o->b; s = o->c; wl = opcost(o);
            } else if (l1 >= 2) {
              int n2 = tt->start[k] - tt->start[k - 1];
              z1 = tt->start[i + 1] + la / n2; z2 = tt->start[k - 1] + la % n2;
              const orc_op *o = &tt->ops[z1], *r = &tt->ops[z2];
              if (o->a != ap) continue;
              u = o->b; up = r->b; s = r->c;
              wl = opcost(o) + mfeE(t, i + 2, k - 2)[o->c * t->sig[k - 1] + r->a] + opcost(r);
            }
            if (wl >= FINF) continue;
            for (int ra = 0; ra < nr; ++ra) {
              int z3 = -1, z4 = -1, v = 0, vp = 0, tb = cp;
              real wr = 0;
              if (l2 == 1) {
                z4 = tt->start[j - 1] + ra;
                const orc_op* o = &tt->ops[z4];
                if (o->c != cp) continue;
                v = vp = o->b; tb = o->a; wr = opcost(o);
              } else if (l2 >= 2) {
                int n2 = tt->start[j] - tt->start[j - 1];
                z3 = tt->start[l + 1] + ra / n2; z4 = tt->start[j - 1] + ra % n2;
                const orc_op *o = &tt->ops[z3], *r = &tt->ops[z4];
                if (r->c != cp) continue;
                vp = o->b; v = r->b; tb = o->a;
                wr = opcost(o) + mfeE(t, l + 2, j - 2)[o->c * t->sig[j - 1] + r->a] + opcost(r);
              }
              if (wr >= FINF) continue;
              for (int xp = 0; xp < 4; ++xp)
                for (int yp = 0; yp < 4; ++yp) {
                  if (!can_pair(m, xp, yp)) continue;
                  real e;
                  if (l1 == 0 && l2 == 0) e = B * (real)m->stack[P][ptype(xp, yp)];
                  else if (l1 == 0 || l2 == 0) e = B * (real)(m->bulge_init[l1 + l2] + (l1 + l2 == 1 ? m->stack[P][ptype(xp, yp)] : 0.0));
                  else e = B * (real)(m->interior_init[l1 + l2] + m->tmm[P][u][v] + m->tmm[ptype(yp, xp)][vp][up]);
                  real val = w0 + e + wl + wr + qin[((s * 4 + xp) * 4 + yp) * St + tb];
                  if (val < bv) { bv = val; bk = 1; bzi = zi; bzj = zj; b1 = z1; b2 = z2; b3 = z3; b4 = z4; bkk = k; bll = l; bxp = xp; byp = yp; bs = s; bt = tb; }
                }
            }
          }
        }
      /* multiloop */
      for (int k = i + 2; k <= j - 1; ++k) {
        const real* A = t->fm[(size_t)(i + 1) * n + (k - 1)];
        const real* Bq = t->fm1[(size_t)k * n + (j - 1)];
        int Sk = t->sig[k], Scq = t->sig[j];
        for (int s = 0; s < Sk; ++s) {
          real val = w0 + B * (real)(m->ml_a + m->ml_c) + A[ap * Sk + s] + Bq[s * Scq + cp];
          if (val < bv) { bv = val; bk = 2; bzi = zi; bzj = zj; bkk = k; bs = s; }
        }
      }
    }
  const orc_op *oi = &tt->ops[bzi], *oj = &tt->ops[bzj];
  int ap = oi->c, cp = oj->a;
  if (bk == 0) {
    const orc_op *o = &tt->ops[b1], *r = &tt->ops[b2];
    c->seq[i + 1] = (uint8_t)o->b; c->seq[j - 1] = (uint8_t)r->b;
    mfe_chain(c, i + 2, j - 2, o->c, r->a);
  } else if (bk == 1) {
    int k = bkk, l = bll, l1 = k - i - 1, l2 = j - l - 1;
    if (l1 == 1) c->seq[i + 1] = (uint8_t)tt->ops[b1].b;
    else if (l1 >= 2) {
      c->seq[i + 1] = (uint8_t)tt->ops[b1].b; c->seq[k - 1] = (uint8_t)tt->ops[b2].b;
      mfe_chain(c, i + 2, k - 2, tt->ops[b1].c, tt->ops[b2].a);
    }
    if (l2 == 1) c->seq[j - 1] = (uint8_t)tt->ops[b4].b;
    else if (l2 >= 2) {
      c->seq[l + 1] = (uint8_t)tt->ops[b3].b; c->seq[j - 1] = (uint8_t)tt->ops[b4].b;
      mfe_chain(c, l + 2, j - 2, tt->ops[b3].c, tt->ops[b4].a);
    }
    mfe_tb_fb(c, k, l, bs, bxp, byp, bt);
  } else {
    mfe_tb_fm(c, i + 1, bkk - 1, ap, bs);
    mfe_tb_fm1(c, bkk, j - 1, bs, cp);
  }
}

static void mfe_tb_fml(mfe_tb* c, int i, int j, int a, int cc) {
  const mfe_tab* t = c->t;
  int n = t->n;
  real gb = (real)t->beta * (real)t->m->ml_b;
  for (;;) {  /* peel leading unpaired positions until the branch starts */
    int Sj1 = t->sig[j + 1], best = -1;
    real bv = t->fm1[(size_t)i * n + j][a * Sj1 + cc];
    if (i + 1 <= j)
      for (int z = t->tt->start[i]; z < t->tt->start[i + 1]; ++z) {
        const orc_op* o = &t->tt->ops[z];
        if (o->a != a) continue;
        real v = gb + opcost(o) + t->fml[(size_t)(i + 1) * n + j][o->c * Sj1 + cc];
        if (v < bv) { bv = v; best = z; }
      }
    if (best < 0) { mfe_tb_fm1(c, i, j, a, cc); return; }
    c->seq[i] = (uint8_t)t->tt->ops[best].b;
    a = t->tt->ops[best].c;
    ++i;
  }
}

static void mfe_tb_fm1(mfe_tb* c, int i, int j, int a, int cc) {
  const mfe_tab* t = c->t;
  int n = t->n;
  real B = (real)t->beta, gb = B * (real)t->m->ml_b, gc = B * (real)t->m->ml_c;
  for (;;) {  /* peel trailing unpaired positions until the closing pair of the branch */
    int Sj1 = t->sig[j + 1], best = -1, bxy = -1;
    real bv = FINF;
    const real* fb = t->fb[(size_t)i * n + j];
    for (int xy = 0; xy < 16; ++xy) {
      real v = gc + fb[(a * 16 + xy) * Sj1 + cc];
      if (v < bv) { bv = v; bxy = xy; }
    }
    if (j - 1 >= i)
      for (int z = t->tt->start[j]; z < t->tt->start[j + 1]; ++z) {
        const orc_op* o = &t->tt->ops[z];
        if (o->c != cc) continue;
        real v = gb + t->fm1[(size_t)i * n + (j - 1)][a * t->sig[j] + o->a] + opcost(o);
        if (v < bv) { bv = v; best = z; }
      }
    if (best < 0) { mfe_tb_fb(c, i, j, a, bxy / 4, bxy % 4, cc); return; }
    c->seq[j] = (uint8_t)t->tt->ops[best].b;
    cc = t->tt->ops[best].a;
    --j;
  }
}

static void mfe_tb_fm(mfe_tb* c, int i, int j, int a, int cc) {
  const mfe_tab* t = c->t;
  int n = t->n, Sj1 = t->sig[j + 1], bk = -1, bs = 0;
  real bv = t->fml[(size_t)i * n + j][a * Sj1 + cc];
  for (int k = i + 1; k <= j; ++k) {
    const real* A = t->fm[(size_t)i * n + (k - 1)];
    const real* Bq = t->fm1[(size_t)k * n + j];
    int Sk = t->sig[k];
    for (int s = 0; s < Sk; ++s) {
      real v = A[a * Sk + s] + Bq[s * Sj1 + cc];
      if (v < bv) { bv = v; bk = k; bs = s; }
    }
  }
  if (bk < 0) { mfe_tb_fml(c, i, j, a, cc); return; }
  mfe_tb_fm(c, i, bk - 1, a, bs);
  mfe_tb_fm1(c, bk, j, bs, cc);
}

/* f_min = min over operator paths and structures of E/kT - sum log x (eq 2.8), and one minimiser (seq, pair; either may be NULL) */
int orc_mfe(const orc_model* m, const orc_tt* tt, int nthreads, double* fmin, uint8_t* seq, int32_t* pair) {
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
  mfe_tab* t = mfe_build(m, tt);
  int n = t->n, cb = 0;
  real best = FINF;
  for (int c = 0; c < t->sig[n]; ++c)
    if (t->fext[n][c] < best) { best = t->fext[n][c]; cb = c; }
  if (fmin) *fmin = (double)best;
  if (seq && pair) {
    mfe_tb tb = {t, seq, pair};
    for (int p = 0; p < n; ++p) { seq[p] = 255; pair[p] = -1; }
    int j = n - 1;
    while (j >= 0) {
      int Sj1 = t->sig[j + 1], bz = -1, bk = -1, bs = 0, bxy = 0;
      real bv = FINF;
      for (int z = tt->start[j]; z < tt->start[j + 1]; ++z) {
        const orc_op* o = &tt->ops[z];
        if (o->c != cb) continue;
        real v = t->fext[j][o->a] + opcost(o);
        if (v < bv) { bv = v; bz = z; }
      }
      for (int k = 0; k <= j - (m->min_hairpin + 1); ++k) {
        const real* fb = t->fb[(size_t)k * n + j];
        for (int s = 0; s < t->sig[k]; ++s)
          for (int xy = 0; xy < 16; ++xy) {
            real v = t->fext[k][s] + fb[(s * 16 + xy) * Sj1 + cb];
            if (v < bv) { bv = v; bz = -1; bk = k; bs = s; bxy = xy; }
          }
      }
      if (bz >= 0) {
        seq[j] = (uint8_t)tt->ops[bz].b;
        cb = tt->ops[bz].a;
        --j;
      } else {
        mfe_tb_fb(&tb, bk, j, bs, bxy / 4, bxy % 4, cb);
        cb = bs;
        j = bk - 1;
      }
    }
  }
  mfe_free(t);
  return 0;
}

/* the definition: enumerate every operator path and every structure, keep the smallest f (tiny designs only) */
typedef struct { const orc_model* m; const orc_tt* tt; int n; uint8_t* seq; int32_t* pair; int* stack; int sp; real cost; real best; double beta;
                 uint8_t* bseq; int32_t* bpair; } bfm_ctx;
static void bfm_structures(bfm_ctx* c, int i) {
  int n = c->n;
  if (i == n) {
    int valid;
    double E = orc_energy(c->m, n, c->seq, c->pair, &valid);
    if (!valid) return;
    real f = c->cost + (real)E * (real)c->beta;
    if (f < c->best) {
      c->best = f;
      if (c->bseq) memcpy(c->bseq, c->seq, n);
      if (c->bpair) memcpy(c->bpair, c->pair, sizeof(int32_t) * n);
    }
    return;
  }
  if (c->sp > 0 && c->stack[c->sp - 1] == i) { --c->sp; bfm_structures(c, i + 1); c->stack[c->sp++] = i; return; }
  c->pair[i] = -1;
  bfm_structures(c, i + 1);
  int lim = c->sp > 0 ? c->stack[c->sp - 1] : n;
  for (int j = i + c->m->min_hairpin + 1; j < lim; ++j) {
    if (!can_pair(c->m, c->seq[i], c->seq[j])) continue;
    c->pair[i] = j; c->pair[j] = i;
    c->stack[c->sp++] = j;
    bfm_structures(c, i + 1);
    --c->sp;
    c->pair[i] = -1; c->pair[j] = -1;
  }
}
static void bfm_paths(bfm_ctx* c, int i, int bond, real cost) {
  if (i == c->n) {
    c->cost = cost;
    for (int p = 0; p < c->n; ++p) c->pair[p] = -1;
    c->sp = 0;
    bfm_structures(c, 0);
    return;
  }
  for (int z = c->tt->start[i]; z < c->tt->start[i + 1]; ++z) {
    const orc_op* o = &c->tt->ops[z];
    if (o->a != bond) continue;
    c->seq[i] = (uint8_t)o->b;
    bfm_paths(c, i + 1, o->c, cost - logl((real)o->x));
  }
}
int orc_brute_force_min(const orc_model* m, const orc_tt* tt, double* fmin, uint8_t* seq, int32_t* pair) {
  int n = tt->n;
  bfm_ctx c;
  memset(&c, 0, sizeof(c));
  c.m = m; c.tt = tt; c.n = n;
  c.seq = (uint8_t*)calloc(n, 1);
  c.pair = (int32_t*)calloc(n, sizeof(int32_t));
  c.stack = (int*)calloc(n + 1, sizeof(int));
  c.beta = 1.0 / model_kT(m);
  c.best = FINF;
  c.bseq = seq; c.bpair = pair;
  bfm_paths(&c, 0, 0, 0.0L);
  if (fmin) *fmin = (double)c.best;
  free(c.seq); free(c.pair); free(c.stack);
  return 0;
}
