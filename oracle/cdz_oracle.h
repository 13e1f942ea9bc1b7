/*
 * cdz_oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, obviously-correct long-double implementation of what the hot path
 * of arXiv 2604.19718 computes, specialised to the nearest-neighbour loop model
 * that BASELINE.json `north_star` fixes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may load this library; it
 * shares no code with paper_2604_19718_b200/csrc.
 *
 * Definition of the result (eqs 2.1-2.4, lines 57-72, bias of line 76):
 *     Z = sum_{phi in Phi(psi)} W(phi) sum_{s in Gamma(phi)} exp(-E(phi,s)/kT),
 *     log Z = -q_psi.
 * W(phi) is the weight of the RNA-sequence tensor train (eq 3.1) in
 * the operator-list encoding of S3c (lines 545-573).
 *
 * Conventions: positions 0..n-1, n = 3L; nucleotides A,C,G,U = 0..3 (line 548);
 * bond sigma_i in [Sigma_i] sits between positions i-1 and i; pair types
 * AU=0 CG=1 GC=2 UA=3 GU=4 UG=5; intervals [i..j] inclusive.
 */
#ifndef CDZ_ORACLE_H
#define CDZ_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  double temperature_K;
  double stack[6][6];      /* [closing pair (phi_i,phi_j)][inner pair (phi_k,phi_l)] */
  double tmm[6][4][4];     /* [pair (phi_a,phi_b)][phi_{a+1}][phi_{b-1}] */
  double hairpin_a, hairpin_b, hairpin_l0; /* H(l) = a + b kT ln(l/l0), l >= min_hairpin */
  double bulge_init[31];   /* index 1..30 */
  double interior_init[31];/* index 2..30, by l1+l2 */
  double ml_a, ml_b, ml_c; /* a + b*unpaired + c*(branches+1) */
  int max_interior;        /* limit on l1+l2 (<=30) */
  int min_hairpin;         /* 3 */
  int allow_all_pairs;     /* test mode: any two nucleotides pair (type 0 tables if not canonical) */
} orc_model;

typedef struct { int a, b, c; double x; } orc_op; /* (a,b,c,x) of PAPER.md lines 547-550 */

typedef struct orc_tt orc_tt;
typedef struct orc_tables orc_tables;

/* ---- tensor train (eqs 3.3/3.4 lines 145-153; S3c.i/ii lines 559-569) ---- */
/* kind 0 = single-codon TT, 1 = codon-pair TT. codon_logw[64] or NULL,
 * pair_logw[64*64] or NULL (log-weight w means factor e^{+w}). */
int  orc_tt_build(const char* aa, int L, int kind, const double* codon_logw,
                  const double* pair_logw, orc_tt** out);
/* same with one codon table per residue, codon_logw_pos[L][64] (line 157: penalty on codon c "at amino acid position i") */
int  orc_tt_build_pos(const char* aa, int L, int kind, const double* codon_logw_pos,
                      const double* pair_logw, orc_tt** out);
int  orc_tt_from_ops(int n, const int* counts, const orc_op* ops, orc_tt** out);
void orc_tt_free(orc_tt* tt);
int  orc_tt_n(const orc_tt* tt);
int  orc_tt_nops(const orc_tt* tt);
void orc_tt_get(const orc_tt* tt, int* sigma /*[n+1]*/, int* counts /*[n]*/, orc_op* ops /*[nops]*/);
/* eq 3.2 (line 137) with open boundaries: log sum_phi W(phi) */
double orc_tt_logsum(const orc_tt* tt);

/* ---- definition-level pieces (brute force) ---- */
/* E(phi,s) in kcal/mol by loop decomposition; *valid=0 if s is not in Gamma(phi). */
double orc_energy(const orc_model* m, int n, const uint8_t* seq, const int32_t* pair, int* valid);
/* log [ W(phi) exp(-E/kT) ], -inf if invalid */
double orc_logweight(const orc_model* m, const orc_tt* tt, const uint8_t* seq, const int32_t* pair);
/* enumerate every operator path (sequence) and every structure. outputs may be NULL.
 * bpp[n*n]: upper triangle P(i.j), diagonal P(i unpaired); base[n*4]; codon[L*64]. */
int orc_brute_force(const orc_model* m, const orc_tt* tt, double* logZ, double* bpp,
                    double* base, double* codon, double* n_states);
/* number of secondary structures (all pairs allowed, hairpin>=min_hairpin, interior<=max_interior) by enumeration */
double orc_count_structures(int n, int min_hairpin, int max_interior);
/* scalar fixed-sequence McCaskill (textbook decomposition), returns log Z */
double orc_mccaskill(const orc_model* m, int n, const uint8_t* seq);

/* ---- the tensor-valued inside recursion ---- */
int  orc_inside(const orc_model* m, const orc_tt* tt, int nthreads, orc_tables** out, double* logZ);
void orc_tables_free(orc_tables* t);
/* copy one cell out as doubles scaled by 2^-shift: which = 0 Qb[a][x][y][c], 1 Qbs, 2 Qm1, 3 Qml, 4 M2, 5 Qm (all [a][c]) */
int  orc_tables_cell(const orc_tables* t, int which, int i, int j, int shift, double* out);
/* log of Qext(j)[c] (natural log; -inf if zero) */
double orc_tables_logqext(const orc_tables* t, int j, int c);

/* ---- stochastic traceback ---- */
int orc_sample(const orc_tables* t, int J, uint64_t seed, uint8_t* seq /*[J][n]*/, int32_t* pair /*[J][n]*/);
/* decision uniform U(seed, sample, kind, i, j) */
double orc_uniform(uint64_t seed, uint64_t sample, uint64_t kind, uint64_t i, uint64_t j);

/* ---- marginals, eqs 2.5-2.7 / 4.1-4.3, by their definitions as constrained sums: one inside pass per pair / nucleotide / codon
 *      (O(n^2) passes: small designs only).  Pinned by the brute-force marginals (tests/test_oracle_pins.py). ---- */
int orc_marginals(orc_tables* t, double* bpp /*[n*n]*/, double* base /*[n*4]*/, double* codon /*[L*64]*/);

/* ---- minimisation, eq 2.8 (line 102), S4d (lines 245-260), Alg S4.5 (lines 706-749): the recursion in the tropical (min, +)
 *      semiring.  f(z, s) = E(phi(z), s)/kT - sum_i log x(z_i) over operator paths z and structures s (units of kT, so
 *      f_min >= -log Z); one minimiser is returned (seq / pair may be NULL).  orc_brute_force_min is the definition by enumeration. */
int orc_mfe(const orc_model* m, const orc_tt* tt, int nthreads, double* fmin, uint8_t* seq /*[n]*/, int32_t* pair /*[n]*/);
int orc_brute_force_min(const orc_model* m, const orc_tt* tt, double* fmin, uint8_t* seq, int32_t* pair);

#ifdef __cplusplus
}
#endif
#endif
