// cdz_internal.h -- host/device structures shared by the translation units of libcdz (CUDA path only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/cdz.h"

#define CDZ_MAX_BOND 8     // bond dimension limit of the kernels
#define CDZ_MAX_STATES 16  // |L_i|, |R_j| limit
#define CDZ_TB 64          // bond-space tile: every position block holds at most CDZ_TB bonds, padded to exactly CDZ_TB
#define CDZ_NCLASS 8       // kernel classes of cdz_profile: 0 gemm, 1 block, 2 rescale, 3 exterior, 4 init, 5 sample
#define CDZ_MAX_SPLIT 16   // split-K limit of the split-point GEMM
#define CDZ_MAX_BATCH 256  // designs advanced together by one launch sequence (larger batches run in chunks)

// ---- Boltzmann factors of the loop model (constant memory image) -------------------------------
struct CModel {
  double wst[6][6];
  double wtm[6][4][4];
  double wbu[32];
  double win[32];
  double wa, wb, wc, wac;
  int max_interior, min_hairpin, allow_all, nps;  // nps = number of pair slots (6 or 16)
  int8_t pslot[16];                               // (x*4+y) -> pair slot or -1
  int8_t ptype[16];                               // (x*4+y) -> pair type for energy lookup
  int8_t slot_x[16], slot_y[16];                  // inverse of pslot
};

struct cdz_model {
  cdz_nn_params p;
  CModel c;
  double kT;
};

// ---- tensor train, host side ---------------------------------------------------------------------
struct cdz_tt {
  int n = 0, kind = -1;
  std::vector<int> sigma;    // [n+1]
  std::vector<int> opstart;  // [n+1]
  std::vector<cdz_op> ops;
  std::vector<int> mid_codon;  // codon index of every middle-base operator, residue by residue in list order (cdz_tt_build only)
  // derived
  int S = 0, LS = 0, RS = 0, MS = 1, maxL = 1, maxR = 1, maxOps = 1;
  std::vector<int> off;                   // [n+2] padded bond offsets: block b owns [b*CDZ_TB, (b+1)*CDZ_TB)
  int NB = 0, sigma_bar = 0;              // number of position blocks; sum_{i<n} Sigma_i
  std::vector<int> blk_start;             // [NB+1] first bond position (0..n) of every block, blk_start[NB] = n+1
  std::vector<int> posblk;                // [n+1] block of bond position i
  std::vector<int> loff, roff;            // [n+1]
  std::vector<uint8_t> ls_a, ls_x;        // [LS]
  std::vector<uint8_t> rs_y, rs_c;        // [RS]
  std::vector<uint8_t> op_l, op_r;        // per operator: local left / right state index
};

// ---- device views --------------------------------------------------------------------------------
struct DevTT {
  int n, S, LS, RS, MS, maxL, maxR, NB;
  const int* blk_start;  // [NB+1]
  const int* posblk;     // [n+1]
  const double* op_x0;   // unscaled operator weights
  const double* Tbar0;   // unscaled transfer matrices
  const int* sig;      // [n+1]
  const int* off;      // [n+2]
  const int* opstart;  // [n+1]
  const uint8_t *op_a, *op_b, *op_c, *op_l, *op_r;
  const int8_t* op_codon;  // codon index (16 b0 + 4 b1 + b2) of a middle-base operator of a cdz_tt_build train, -1 otherwise
  double* op_x;        // scaled operator weights
  const int* loff;     // [n+1]
  const int* roff;     // [n+1]
  const uint8_t *ls_a, *ls_x, *rs_y, *rs_c;
  const int8_t* lsidx;  // [n][MS][4]: local index of left state (a,x) at a position, -1 if absent
  const int8_t* rsidx;  // [n][4][MS]: local index of right state (y,c)
  const int* bondpos;  // [S+1?] position of each bond index (as left bond of that position), bondpos[off[i]+a] = i
  const int* lspos;    // [LS]
  const int* rspos;    // [RS]
  double* Tbar;        // [n][MS*MS], scaled
  const double* wh;    // [n+1] hairpin Boltzmann factor by loop length
};

// All tables are square row-major matrices over the packed index spaces (bonds S, left states LS, right
// states RS); cell (i,j) occupies the block rows(i) x cols(j).
template <typename T>
struct DevTabT {
  T *QB;    // LS x RS : Qb(i,j)[l][r]
  T *DD;    // LS x RS : mismatch-dressed extension of Qb(k,l), stored at cell (k-1,l+1)
  T *D1;    // LS x S  : DD summed over the right nucleotide
  T *D2T;   // RS x S  : DD summed over the left nucleotide, transposed: row (l+1; v',t), column (k-1, s)
  T *GI;    // S  x S  : DD summed over both
  T *QBS;   // S x S
  T *QM;    // S x S   : row (i,a), column (j+1,c)
  T *QM1T;  // S x S   : transposed: row (j+1,c), column (i,a)
  T *QML;   // S x S
  T *M2;    // S x S
  T *EM;    // S x S   : E(i,j) = Tbar_i..Tbar_j; the diagonal holds E(i,i-1) = identity
  T *EMT;   // S x S   : EM transposed (row (j+1,c), column (i,a))
  T *QBST;  // S x S   : QBS transposed
  T *XE;    // S x S   : XE(i,j) = sum_u w_In(u) X_u(i,j) + w_H(d-1) E(i+2,j-2), row (i+2, a2), column (j-1, c2): the loop body between the two
            //           closing-mismatch positions of cell (i,j) (read by the outside pass for the operator usages)
  T *XS;    // [n][27][MS*MS] : interior-loop bodies X_u(i0,j), u = 4..30, of the top row of the last block of every column j
  T *Qext;  // [n+1][MS]
  T *GP;    // split-point GEMM partial sums: [block row I][split][CDZ_TB*CDZ_TB]
  T *R;     // [S] exterior accumulator
  int* scale;    // [n+2] prefix sums P of the per-position scale bits s_m (true = stored * 2^{P[j+1]-P[i]})
  int* dP;       // [n+2] increment of P decided by the last rescale event
  int* EB;       // [S]  dP at the position of every bond index
  int* EL;       // [LS] dP at the position of every left state
  int* ER;       // [RS] dP at (position + 1) of every right state
  int* eA;       // [S] CDZ_FP32_SCALED: binary exponent of the largest finished entry of every QM row (row scale of the fp32 contraction)
  int* eB;       // [S] the same for the rows of QM1T
  int* ctrl;     // control block: [0]=n_rescales [1]=overflow flag [2]=max |exponent| seen at an event
  double* result; // [0]=logZ [1]=Z mantissa [2]=log scale
};
typedef DevTabT<double> DevTab;

struct Ctx {
  DevTT tt;
  DevTab tab;
  const CModel* cm;  // Boltzmann tables (device copy inside the workspace)
  Ctx* batch;        // [CDZ_MAX_BATCH] scratch for the handle array of a batched launch
};

struct cdz_tables {
  const cdz_model* model = nullptr;
  const cdz_tt* tt = nullptr;
  int precision = CDZ_FP64;
  cudaStream_t stream = nullptr;
  cudaStream_t marg_stream = nullptr;  // stream of the last cdz_marginals call
  void* base = nullptr;  // device allocation (owned if owns_base)
  bool owns_base = false;
  size_t bytes = 0;
  Ctx h;         // host copy of the device view
  Ctx* d_ctx = nullptr;  // device copy (inside base)
  int n_rescales = 0;
  int rescale_first = 1;  // rescale events after block diagonals rescale_first * 2^k (cdz_debug_set_rescale_start)
  // per-kernel-class device times of the last pass (cdz_set_profiling): events between consecutive launches
  bool profile = false;
  std::vector<cudaEvent_t> evs;
  std::vector<int> ev_class;
  size_t nev_inside = 0;  // events recorded by the last inside pass (later calls append after them, never beyond one call's worth)
  long launches[CDZ_NCLASS] = {0, 0, 0, 0, 0, 0, 0, 0};
  double inside_ms = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool done = false;
};

// number of K-splits of the split-point GEMM on block diagonal D (B designs advanced together)
inline int cdz_nsplit(int NB, int D, int B) {
  if (D < 2) return 0;
  // 64x64 tiles, 3 CTAs per SM by shared memory: one wave = 444 CTAs.  With s splits the launch takes
  // ceil(nblk * s / 444) waves of K/s each: take the s <= 16 that minimises waves / s (smallest s on ties).
  const int nblk = (NB - D) * B, ks = D - 1;
  int best = 1;
  double bestc = 1e30;
  for (int s = 1; s <= CDZ_MAX_SPLIT && s <= ks; ++s) {
    const double c = (double)((nblk * s + 443) / 444) / (double)s;
    if (c < bestc - 1e-12) { bestc = c; best = s; }
  }
  return best;
}

// ---- internal entry points -----------------------------------------------------------------------
void cdz_set_error(const std::string& s);
struct cdz_cell_cfg { int M, ML, MR, nps, maxpos, span, C; size_t smem; };
int cdz_cell_config(cdz_tables* const* ts, int B, cdz_cell_cfg* cfg);
void cdz_launch_cells(const Ctx* d_ctxs, int B, int nblk, int D, int nsplit, const cdz_cell_cfg* cfg, cudaStream_t st);
int cdz_launch_inside(cdz_tables* const* ts, int B, cudaStream_t st);
int cdz_wait_pass(cdz_tables* t, cudaStream_t st);
int cdz_launch_sample(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, cudaStream_t st);

#define CDZ_CUDA(call)                                                                       \
  do {                                                                                       \
    cudaError_t e__ = (call);                                                                \
    if (e__ != cudaSuccess) {                                                                \
      cdz_set_error(std::string(#call) + ": " + cudaGetErrorString(e__));                    \
      return CDZ_ECUDA;                                                                      \
    }                                                                                        \
  } while (0)
