/*
 * cdz.h -- C ABI of the B200 (sm_100a) codon-design inside-pass library.
 *
 * Hot path of arXiv 2604.19718 ("Direct RNA sequence design under codon constraints
 * using expressive tensor-based secondary structure models"), specialised as
 * BASELINE.json `north_star` fixes it: the tensor-valued inside (partition-function)
 * recursion over all coding sequences Phi(psi) (eqs 2.1-2.4, lines 57-72)
 * and all unpseudoknotted structures, with a McCaskill-style nearest-neighbour loop
 * model; sequence summation enters through the RNA-sequence tensor train (eq 3.1,
 * line 131) exactly as in chi-hat (eq 3.8).
 *
 * Conventions
 *   positions 0..n-1 (n = 3L); nucleotides A,C,G,U = 0..3 (line 548); codon index
 *   16*b0 + 4*b1 + b2; pair types AU=0 CG=1 GC=2 UA=3 GU=4 UG=5.
 *   Pointers named *_dev are CUDA device pointers, all others are host pointers.
 *   `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   All functions return 0 on success or a negative cdz_status; the text of the
 *   last error of the calling thread is available from cdz_last_error().
 *   Handles are created by the library, owned by the caller and released with the
 *   matching *_destroy.  The library never falls back to a CPU implementation.
 */
#ifndef CDZ_H
#define CDZ_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CDZ_OK = 0,
  CDZ_EINVAL = -1,    /* bad argument, unknown residue, non-finite weight */
  CDZ_ENOMEM = -2,    /* host or device allocation failed / workspace too small */
  CDZ_ECUDA = -3,     /* a CUDA runtime call or kernel failed */
  CDZ_EOVERFLOW = -4, /* dynamic range left the representable window despite rescaling */
  CDZ_ESTATE = -5     /* call order (e.g. sampling before the inside pass finished) */
} cdz_status;

enum { CDZ_TT_SINGLE_CODON = 0, CDZ_TT_CODON_PAIR = 1 };
/* CDZ_FP64: everything in fp64 (tolerance 1e-9 relative in log Z).
 * CDZ_FP32_SCALED (BASELINE.json configs[2], "single precision", line 622 row renormalisation): the split-point
 * contraction -- the O(n^3) part -- runs in single precision on the tensor cores (3 x TF32 split operands, fp32 accumulation) with
 * an exact power-of-two scale per operand row, re-decided every block diagonal; tables, loop terms, scale bookkeeping and the
 * exterior sum stay fp64.  Tolerance 1e-4 relative in log Z.  All designs of a batch share one precision. */
enum { CDZ_FP64 = 0, CDZ_FP32_SCALED = 1 };

/* Nearest-neighbour loop model (BASELINE.json configs[0]); energies in kcal/mol.
 *   hairpin(l)  = hairpin_a + hairpin_b * kT * ln(l / hairpin_l0) + tmm[p(i,j)][phi_{i+1}][phi_{j-1}],  l >= min_hairpin
 *   stack       = stack[p(i,j)][p(k,l)]            closing pair (phi_i,phi_j), inner pair (phi_k,phi_l)
 *   bulge(l)    = bulge_init[l] (+ stack[..] if l == 1),  1 <= l <= max_interior
 *   interior    = interior_init[l1+l2] + tmm[p(i,j)][phi_{i+1}][phi_{j-1}] + tmm[p(l,k)][phi_{l+1}][phi_{k-1}]
 *   multiloop   = ml_a + ml_b * unpaired + ml_c * (branches + 1);   exterior loop = 0
 * kT = R * temperature_K, R = 8.31446261815324/4184 kcal/(mol K).  No symmetry is enforced. */
typedef struct {
  double temperature_K;
  double stack[6][6];
  double tmm[6][4][4];
  double hairpin_a, hairpin_b, hairpin_l0;
  double bulge_init[31];    /* index 1..30 */
  double interior_init[31]; /* index 2..30 */
  double ml_a, ml_b, ml_c;
  int32_t max_interior;     /* <= 30 */
  int32_t min_hairpin;      /* >= 3 */
  int32_t allow_all_pairs;  /* test mode: any two nucleotides may pair (non-canonical use pair type 0) */
} cdz_nn_params;

/* One tensor-train operator (a,b,c,x) of PAPER.md S3c (lines 545-557):
 * T_i[a,b,c] += x, a in [Sigma_i], b a nucleotide, c in [Sigma_{i+1}], x > 0. */
typedef struct { int32_t a, b, c; double x; } cdz_op;

typedef struct cdz_model cdz_model;
typedef struct cdz_tt cdz_tt;
typedef struct cdz_tables cdz_tables;

/* Result / accounting record filled by cdz_tables_info (host). */
typedef struct {
  int32_t n;                /* nucleotides */
  int32_t sigma_bar;        /* sum_{i<n} Sigma_i */
  int32_t n_left_states;    /* sum_i |L_i|, distinct (sigma_i, phi_i) */
  int32_t n_right_states;   /* sum_j |R_j|, distinct (phi_j, sigma_{j+1}) */
  int32_t precision;
  int32_t n_rescales;       /* dynamic rescale events during the pass */
  double n_cc;              /* structurally non-zero split-point terms (i,k,j) */
  double n_loop;            /* one-inner-pair terms (i,j,l1,l2) */
  double split_mac;         /* exact multiply-adds of the split-point contraction */
  double table_bytes;       /* device bytes held by the handle */
  double bytes_per_cell;    /* table_bytes / (n(n+1)/2) */
  double log_scale;         /* sum_m s_m ln 2 added back into log Z */
  double inside_ms;         /* device time of the last inside pass (CUDA events) */
} cdz_info;

const char* cdz_last_error(void);
int cdz_version(void);

/* ---- model ---------------------------------------------------------------- */
int cdz_model_create(const cdz_nn_params* params, cdz_model** out);
void cdz_model_destroy(cdz_model* m);

/* ---- tensor train (host, O(n)) -------------------------------------------- */
/* Codon tensor train of an amino-acid string aa[0..L) over "ACDEFGHIKLMNPQRSTVWY".
 *   kind = CDZ_TT_SINGLE_CODON: eq 3.4 (line 151), operator lists of S3c.i (lines 559-563);
 *   kind = CDZ_TT_CODON_PAIR  : eq 3.3 (line 145) in the S3c.ii form (lines 565-569).
 * codon_logw: [64] (or NULL): factor e^{+w} on the middle-base operator of that codon (line 157).
 * pair_logw : [64*64] row = 5' codon (or NULL; CODON_PAIR only): factor on the 5'-base operator (line 163).
 * Open chain: Sigma_0 = 1, the last bond is summed out. */
int cdz_tt_build(const char* aa, int L, int kind, const double* codon_logw, const double* pair_logw, cdz_tt** out);
/* Same with one codon table per residue, codon_logw_pos[L][64]: the paper's soft constraint penalises codon c "at amino acid
 * position i" (line 157); row k applies to residue k only.  NULL = no codon weights. */
int cdz_tt_build_pos(const char* aa, int L, int kind, const double* codon_logw_pos, const double* pair_logw, cdz_tt** out);
/* Generic operator lists (lines 545-557, noncoding bases line 573). counts[n], ops[sum counts]. Bond dims <= 8. */
int cdz_tt_from_operators(int n, const int32_t* counts, const cdz_op* ops, cdz_tt** out);
void cdz_tt_destroy(cdz_tt* tt);
int cdz_tt_length(const cdz_tt* tt);
/* sigma[n+1], counts[n] (either may be NULL); returns total operator count */
int cdz_tt_describe(const cdz_tt* tt, int32_t* sigma, int32_t* counts);

/* ---- inside pass (device) -------------------------------------------------- */
/* Device bytes cdz_inside needs for (tt, precision); the caller may allocate them
 * (e.g. as a torch uint8 tensor) and pass the pointer as workspace_dev. */
int cdz_workspace_bytes(const cdz_tt* tt, int precision, size_t* bytes);
/* Runs the whole inside recursion (all anti-diagonals, exterior, log Z) asynchronously on `stream`.
 * workspace_dev may be NULL (the library allocates and owns the tables) or a device
 * buffer of >= cdz_workspace_bytes bytes that must outlive the handle.
 * logZ_host (may be NULL) is written by a host-side epilogue after the pass: the call
 * synchronises `stream` only if logZ_host != NULL; otherwise use cdz_tables_logz. */
int cdz_inside(const cdz_model* m, const cdz_tt* tt, int precision, void* workspace_dev, size_t workspace_bytes,
               void* stream, cdz_tables** out, double* logZ_host);
/* B independent designs advanced together (BASELINE.json configs[4]); workspace_dev[b] may be NULL. */
int cdz_inside_batch(const cdz_model* m, const cdz_tt* const* tts, int B, int precision, void* const* workspace_dev,
                     const size_t* workspace_bytes, void* stream, cdz_tables** out, double* logZ_host);
/* Re-run the pass on an existing handle (same tt/model); used by the timing harness. */
int cdz_inside_rerun(cdz_tables* t, void* stream);
int cdz_inside_rerun_batch(cdz_tables* const* t, int B, void* stream);
/* Synchronises the handle's stream and returns log Z = -q_psi (eq 2.4). */
int cdz_tables_logz(cdz_tables* t, double* logZ_host);
int cdz_tables_info(cdz_tables* t, cdz_info* info);
void cdz_tables_destroy(cdz_tables* t);
/* Kernel accounting of the last pass on this handle.  cdz_set_profiling(t, 1) makes the next passes record a CUDA
 * event between consecutive launches on the pass's stream; cdz_profile then synchronises the stream and returns, per
 * kernel class (0 split-point GEMM, 1 block/cell kernel, 2 rescale, 3 exterior, 4 init, 5 traceback; [8] each),
 * the summed device milliseconds (0 when profiling was off) and the launch counts (always counted). */
int cdz_set_profiling(cdz_tables* t, int on);
int cdz_profile(cdz_tables* t, double* ms_out, int64_t* launches_out);
/* Parity knob: the per-position scales are re-decided after block diagonals first, 2 first, 4 first, ... (default first = 1).
 * Power-of-two scales make log Z independent of the schedule up to rounding; the tests move the events to check exactly that
 * (SURVEY 8c "scaling-schedule invariance").  Takes effect at the next cdz_inside_rerun of the handle. */
int cdz_debug_set_rescale_start(cdz_tables* t, int first);
/* Debug / parity access: copy one cell to host as doubles (true value * 2^-shift_out).
 * which: 0 Qb as [a][x][y][c] dense, 1 Qbs, 2 Qm1, 3 Qml, 4 M2, 5 Qm (all [a][c]). Returns element count. */
int cdz_tables_cell(cdz_tables* t, int which, int i, int j, double* out_host, int* shift_out);
/* log Qext(j)[c] (natural log, scale included) */
int cdz_tables_logqext(cdz_tables* t, int j, int c, double* out_host);

/* ---- exact Boltzmann samples (device) ------------------------------------- */
/* J i.i.d. samples (phi, s) ~ W(phi) exp(-E/kT) / Z by stochastic traceback (PAPER.md S4c,
 * Alg S4.4; decision order in DESIGN.md).  seq_dev [J][n] uint8 (0..3),
 * pair_dev [J][n] int32 partner or -1.  Uniforms are U(seed, sample, kind, i, j). */
int cdz_sample(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, void* stream);

/* cdz_sample for callers that must not allocate device memory (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same kernel, bit-identical samples for the same (tables, J, seed).  The traceback stacks, the
 * only scratch of the sampler (n/4 + 16 items of 20 bytes per sample), live in a static device array of
 * CDZ_NOALLOC_STACK_ITEMS items (8.0 MB) that every GPU loading the library holds until the process exits, instead of a
 * stream-ordered allocation.  The call makes no cudaMalloc / cudaFree / cudaMallocAsync and creates no events.
 * Limit: J * (n/4 + 16) <= CDZ_NOALLOC_STACK_ITEMS (J <= 106 at n = 15000, J <= 3125 at n = 450); CDZ_EINVAL with a message
 * beyond it (use cdz_sample).  All calls on one GPU share the array: calls that overlap on the GPU (two streams, two host
 * threads) race; serialise them.  The array keeps the previous call's contents and needs no clearing (every item is written
 * before it is read).  Asynchronous on `stream`; seq_dev / pair_dev are caller-owned as in cdz_sample. */
#define CDZ_NOALLOC_STACK_ITEMS 400000
int cdz_sample_noalloc(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, void* stream);

/* ---- marginals (device) ---------------------------------------------------- */
/* Outside (adjoint) pass over the tables of a finished inside pass: the paper's ComputeReverse (Alg S4.3) as the
 * reverse-mode adjoint of the recursion.  Asynchronous on `stream` (it waits for the inside pass by an event
 * if that ran on another stream); outputs are valid after the stream has been synchronised.  Every output may be NULL:
 *   bpp_dev   [n][n] doubles, fully overwritten: upper triangle P(i.j) (eq 2.5 line 85, eq 4.1), diagonal P(i unpaired)
 *             (computed from the unpaired operator usages, NOT as 1 - row sum), lower triangle 0;
 *   base_dev  [n][4]  P(phi_m = b), eq 2.6 line 90 / eq 4.2;
 *   codon_dev [L][64] p_k(c), c = 16 b0 + 4 b1 + b2, eq 2.7 line 96 / eq 4.3; exactly 0 on codons that do not encode
 *             residue k.  Needs a tensor train from cdz_tt_build / cdz_tt_build_pos (CDZ_EINVAL for generic operator lists).
 * workspace_dev: device buffer of >= cdz_marginals_workspace_bytes bytes, caller-owned, or NULL (the library then takes and
 * returns the memory with the stream-ordered allocator; CDZ_ENOMEM if it does not fit).  No host synchronisation either way.
 * CDZ_ESTATE before cdz_inside. */
int cdz_marginals_workspace_bytes(const cdz_tables* t, size_t* bytes);
int cdz_marginals(cdz_tables* t, void* workspace_dev, size_t workspace_bytes, double* bpp_dev, double* base_dev,
                  double* codon_dev, void* stream);
/* Synchronises the stream of the last cdz_marginals call and reports its device-side checks: CDZ_EOVERFLOW when an operator
 * usage left [0,1] or the usages at some position do not sum to 1 within 1e-6 (non-finite values included), else CDZ_OK. */
int cdz_marginals_status(cdz_tables* t);

/* ---- fixed-sequence evaluation of sampled sequences (PAPER.md S4f line 779) ---- */
/* For J sequences seq_host[J][n] (nucleotides 0..3, host) -- typically the output of cdz_sample -- computes with the same kernels
 *   logZ_host[J]      log Z(phi) of the fixed sequence under the loop model (= -q(phi); ordinary McCaskill), required;
 *   logW_host[J]      log W(phi), the sequence's weight in the design's tensor train (-inf if phi is outside the design space);
 *                     NULL or needs `design`;
 *   unpaired_host[J][n]  P(i unpaired | phi) from the outside pass; NULL to skip.
 * Each sequence is the tensor train with one operator (0, phi_i, 0, 1) per position (lines 545-557); the sequences are advanced
 * together in chunks by cdz_inside_batch (chunk size from the free device memory, at most max_batch if max_batch > 0).
 * Blocking: returns after the results are in the host buffers.  Tables are created and released inside the call. */
int cdz_eval_sequences(const cdz_model* m, const cdz_tt* design, int n, int J, const uint8_t* seq_host, int max_batch,
                       double* logZ_host, double* logW_host, double* unpaired_host, void* stream);

/* ---- minimisation (eq 2.8, S4d lines 245-260, Alg S4.5) ---- */
/* The recursion in the tropical (min, +) semiring: fmin_host = min over operator paths z (one operator per position, bonds matching)
 * and structures s of  f(z, s) = E(phi(z), s)/kT - sum_i log x(z_i)  (units of kT; fmin >= -log Z), and one minimiser:
 * seq_dev [n] uint8 (0..3), pair_dev [n] int32 (partner or -1); both NULL to skip the traceback.  workspace_dev: a device buffer of
 * >= cdz_workspace_bytes(tt, CDZ_FP64) bytes or NULL (library allocation); the tropical tables live in it during the call only.
 * Blocking: returns after fmin_host has been written.  Ties between minimisers are broken by the enumeration order. */
int cdz_mfe(const cdz_model* m, const cdz_tt* tt, void* workspace_dev, size_t workspace_bytes, void* stream, double* fmin_host,
            uint8_t* seq_dev, int32_t* pair_dev);

/* ---- frequency matching (PAPER.md S4e lines 751-771, Alg S4.6) ---- */
/* Finds per-codon bonuses f (log f = a codon_logw table for cdz_tt_build) such that the accumulated exact codon marginals of the design
 * distribution, b[c] = sum_k p_k(c), match the target frequencies bstar[c] = sum_{k: c codes aa_k} fstar_c / sum_{c' codes aa_k} fstar_c'
 * (the frequencies of the structure-free uniform distribution with bonuses fstar = exp(logf_star), as in Alg S4.6).  Fixed-point iteration
 * f <- f bstar / b from f = fstar, stopped when || log(b / bstar) ||_inf < rtol (the paper uses 0.002) or after max_iter iterations; anderson != 0
 * applies Anderson acceleration over the whole history (line 771).  Every iteration is cdz_tt_build + cdz_inside + cdz_marginals on
 * the device.  logf_out[64]: final log-bonuses; err_history[max_iter] (may be NULL): the error of every evaluated iterate;
 * n_iter_out: number of evaluated iterates.  pair_logw as in cdz_tt_build.  Blocking.  Not converged is not an error: check err_history. */
int cdz_match_frequencies(const cdz_model* m, const char* aa, int L, int kind, const double* logf_star, const double* pair_logw,
                          double rtol, int max_iter, int anderson, double* logf_out, double* err_history, int* n_iter_out,
                          void* stream);

/* ---- the paper's tensor-based free-energy model (PAPER.md S2b lines 430-437; eqs 3.5-3.8; Alg S4.1 / S4.2 lines 586-622) ---- */
/* Parameters (host pointers, read during the call only): gamma = model dimension (<= 8), xi = number of pair conformations (<= 4),
 *   V [4][gamma][gamma]           matrix of an unpaired base x (eq 3.6, second case),
 *   B [4][4][xi][gamma][gamma]    B[x][y][rho] = tensor of the 5' side of a pair with 5' base x and 3' base y ("B_{i,j}^rho"); B[y][x][rho] is the
 *                                 tensor of its 3' side ("B_{j,i}^rho"); all-zero B[x][y] = x.y cannot pair,
 *   S [gamma][gamma]              weighted trace Tr_S[X] = Tr[S X] (line 178),
 * min_hairpin: a pair k.l needs l - k - 1 >= min_hairpin (line 483: 3).  All entries finite and >= 0.  Limits of this version:
 * gamma x (largest bond dimension of tt) <= 32 and (number of pairable (x,y)) x xi x bond x (96 / gamma) <= 6144; CDZ_EINVAL beyond. */
typedef struct {
  int32_t gamma, xi, min_hairpin;
  const double* V;
  const double* B;
  const double* S;
} cdz_tm_params;
typedef struct {
  double device_ms;        /* device time of the full-size pass (CUDA events on `stream`: table clear, all block diagonals, final trace) */
  double gemm_ms;          /* of which: the tensor-core tile kernels (tm_gemm_kernel) */
  double block_ms;         /* of which: the per-block kernels (chi-hat + in-block edges, tm_block_kernel) */
  double gemm_flop;        /* FLOP of the tensor-core tiles: 2 x 64^3 x (number of K blocks), padding included */
  double table_bytes;      /* the two S x S tables */
  int64_t launches, gemm_launches;
  int32_t S, NB;           /* flattened (block-padded) dimension sum_i gamma Sigma_i and its number of 64-blocks */
  double scale_rate;       /* r: the operator weights of position q were multiplied by 2^-(P[q+1] - P[q]), P[q] = floor(q r); log Z = log Z_stored + P[n] ln 2 */
} cdz_tm_info;
/* log Z = -q_psi (eq 2.4 line 72) of the design distribution under the tensor model: the sum over every operator path (coding sequence,
 * weights included) of `tt` and every unpseudoknotted structure of the state's tensor diagram (eq S2.1), by the recursion
 *   Q_{i,j} = sum_{k in [i:j)} Q_{i,k} Q_{j,k}^T (i < j),  Q_{j,k} = chi-hat_{k,j}(Q_{k+1,j-1}) (j > k),  Z = sum_{sigma_n} Tr_S[Q_{0,n}]
 * run as a block wavefront with fp64 tensor-core tiles (csrc/cdz_tm.cu).  Open chain as in cdz_tt_build.  workspace_dev: a device
 * buffer of >= cdz_tm_workspace_bytes bytes (it then holds the tables after the call: cdz_tm_block) or NULL (allocated and freed
 * inside).  Blocking: returns after logZ_host has been written.  info may be NULL.  CDZ_EOVERFLOW if Z leaves the fp64 range in the
 * stored scale (power-of-two scales per position at a uniform rate, measured by pilot passes over the first 60 and 600 positions). */
int cdz_tm_workspace_bytes(const cdz_tm_params* p, const cdz_tt* tt, size_t* bytes);
int cdz_tm_inside(const cdz_tm_params* p, const cdz_tt* tt, void* workspace_dev, size_t workspace_bytes, void* stream, double* logZ_host,
                  cdz_tm_info* info);
/* Debug / parity access to the tables a cdz_tm_inside call left in a caller workspace (same p, tt; scale_rate from its info):
 * which = 0: the upper block Q_{i,j}, 0 <= i <= j <= n, as [gamma Sigma_i][gamma Sigma_j]; which = 1: the lower block Q_{j,i}, i < j, as
 * [gamma Sigma_j][gamma Sigma_i] (index (sigma, zeta) -> sigma gamma + zeta, line 211).  true value = out x 2^shift_out.  Returns the
 * element count. */
int cdz_tm_block(const cdz_tm_params* p, const cdz_tt* tt, const void* workspace_dev, double scale_rate, int which, int i, int j,
                 double* out_host, int* shift_out);

/* J exact samples (sequence, structure) ~ W(phi) Z(phi, s) / Z under the tensor model (section 4a) by stochastic traceback of
 * the tables a cdz_tm_inside call left in a caller workspace (same p, tt): one warp per sample, the alternatives of Alg S4.4 (lines 657-701)
 * in the fixed order of DESIGN.md section 17, uniforms U(seed, sample, kind, i, j) with kinds 16-19.  seq_dev [J][n] uint8 (0..3),
 * pair_dev [J][n] int32 partner or -1.  Asynchronous on `stream` (the stacks are a stream-ordered allocation). */
int cdz_tm_sample(const cdz_tm_params* p, const cdz_tt* tt, void* workspace_dev, int J, uint64_t seed, uint8_t* seq_dev,
                  int32_t* pair_dev, void* stream);

/* ---- convenience: host buffers end to end (used for the e2e timing) -------- */
/* Builds nothing: runs cdz_inside_rerun, samples J states and copies them to host buffers. */
int cdz_run_host(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_host, int32_t* pair_host, double* logZ_host,
                 void* stream);

#ifdef __cplusplus
}
#endif
#endif
