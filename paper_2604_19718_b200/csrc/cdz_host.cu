// cdz_host.cu -- host side of libcdz: error state, loop-model tables, tensor-train builder, table handles.
// (CUDA path; shares nothing with oracle/.)
#include <math.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <new>

#include "cdz_internal.h"
#include "cdz_outside.h"

static thread_local std::string g_err;
void cdz_set_error(const std::string& s) { g_err = s; }
extern "C" const char* cdz_last_error(void) { return g_err.c_str(); }
extern "C" int cdz_version(void) { return 1; }

// ------------------------------------------------------------------------------------------------
// model: Boltzmann factors exp(-E/kT) of every loop table (BASELINE.json configs[0])
// ------------------------------------------------------------------------------------------------
static const double kGasR = 8.31446261815324 / 4184.0;  // kcal/(mol K)

extern "C" int cdz_model_create(const cdz_nn_params* p, cdz_model** out) {
  if (!p || !out) { cdz_set_error("cdz_model_create: null argument"); return CDZ_EINVAL; }
  if (!(p->temperature_K > 0) || p->max_interior < 0 || p->max_interior > 30 || p->min_hairpin < 3 ||
      !(p->hairpin_l0 > 0)) {
    cdz_set_error("cdz_model_create: need T>0, 0<=max_interior<=30, min_hairpin>=3, hairpin_l0>0");
    return CDZ_EINVAL;
  }
  const double* raw = reinterpret_cast<const double*>(p);
  for (size_t k = 0; k < offsetof(cdz_nn_params, max_interior) / sizeof(double); ++k)
    if (!std::isfinite(raw[k])) { cdz_set_error("cdz_model_create: non-finite parameter"); return CDZ_EINVAL; }
  cdz_model* m = new (std::nothrow) cdz_model;
  if (!m) return CDZ_ENOMEM;
  m->p = *p;
  m->kT = kGasR * p->temperature_K;
  const double beta = 1.0 / m->kT;
  CModel& c = m->c;
  memset(&c, 0, sizeof(c));
  for (int a = 0; a < 6; ++a) {
    for (int b = 0; b < 6; ++b) c.wst[a][b] = exp(-p->stack[a][b] * beta);
    for (int x = 0; x < 4; ++x)
      for (int y = 0; y < 4; ++y) c.wtm[a][x][y] = exp(-p->tmm[a][x][y] * beta);
  }
  for (int l = 1; l <= 30; ++l) c.wbu[l] = exp(-p->bulge_init[l] * beta);
  for (int l = 2; l <= 30; ++l) c.win[l] = exp(-p->interior_init[l] * beta);
  c.wa = exp(-p->ml_a * beta);
  c.wb = exp(-p->ml_b * beta);
  c.wc = exp(-p->ml_c * beta);
  c.wac = c.wa * c.wc;
  c.max_interior = p->max_interior;
  c.min_hairpin = p->min_hairpin;
  c.allow_all = p->allow_all_pairs ? 1 : 0;
  // pair slots: canonical pairs in (x,y)-lexicographic order, all 16 combinations in test mode
  static const int canon[4][4] = {{-1, -1, -1, 0}, {-1, -1, 1, -1}, {-1, 2, -1, 4}, {3, -1, 5, -1}};
  int ns = 0;
  for (int x = 0; x < 4; ++x)
    for (int y = 0; y < 4; ++y) {
      int t = canon[x][y];
      c.ptype[x * 4 + y] = (int8_t)(t >= 0 ? t : 0);
      if (t >= 0 || c.allow_all) {
        c.pslot[x * 4 + y] = (int8_t)ns;
        c.slot_x[ns] = (int8_t)x;
        c.slot_y[ns] = (int8_t)y;
        ++ns;
      } else {
        c.pslot[x * 4 + y] = -1;
      }
    }
  c.nps = ns;
  *out = m;
  return CDZ_OK;
}
extern "C" void cdz_model_destroy(cdz_model* m) { delete m; }

// ------------------------------------------------------------------------------------------------
// tensor train builder (eqs 3.3/3.4 lines 145-153, operator lists S3c lines 545-573)
// ------------------------------------------------------------------------------------------------
namespace {
struct AminoCodons { char aa; const char* codons; };
// standard genetic code, sense codons only (the listing of), RNA alphabet
const AminoCodons kCode[20] = {
    {'A', "GCA GCC GCG GCU"}, {'C', "UGC UGU"}, {'D', "GAC GAU"}, {'E', "GAA GAG"}, {'F', "UUC UUU"},
    {'G', "GGA GGC GGG GGU"}, {'H', "CAC CAU"}, {'I', "AUA AUC AUU"}, {'K', "AAA AAG"},
    {'L', "CUA CUC CUG CUU UUA UUG"}, {'M', "AUG"}, {'N', "AAC AAU"}, {'P', "CCA CCC CCG CCU"},
    {'Q', "CAA CAG"}, {'R', "AGA AGG CGA CGC CGG CGU"}, {'S', "AGC AGU UCA UCC UCG UCU"},
    {'T', "ACA ACC ACG ACU"}, {'V', "GUA GUC GUG GUU"}, {'W', "UGG"}, {'Y', "UAC UAU"}};

int nuc_of(char ch) { return ch == 'A' ? 0 : ch == 'C' ? 1 : ch == 'G' ? 2 : ch == 'U' ? 3 : -1; }

// codon indices (16 b0 + 4 b1 + b2), ascending, for one residue; empty if unknown
std::vector<int> codon_set(char aa) {
  std::vector<int> v;
  for (const auto& e : kCode)
    if (e.aa == aa)
      for (const char* s = e.codons; *s;) {
        v.push_back(16 * nuc_of(s[0]) + 4 * nuc_of(s[1]) + nuc_of(s[2]));
        s += 3;
        if (*s == ' ') ++s;
      }
  std::sort(v.begin(), v.end());
  return v;
}

// compact ascending ranks of the values that occur
std::map<int, int> rank_map(const std::vector<int>& vals) {
  std::map<int, int> r;
  for (int v : vals) r[v] = 0;
  int k = 0;
  for (auto& kv : r) kv.second = k++;
  return r;
}

int finalize_tt(cdz_tt* tt) {
  const int n = tt->n;
  tt->MS = 1;
  tt->sigma_bar = 0;
  for (int i = 0; i <= n; ++i) {
    tt->MS = std::max(tt->MS, tt->sigma[i]);
    if (i < n) tt->sigma_bar += tt->sigma[i];
  }
  if (tt->MS > CDZ_MAX_BOND) { cdz_set_error("tensor train bond dimension exceeds 8"); return CDZ_EINVAL; }
  if (tt->sigma[0] != 1) { cdz_set_error("Sigma_0 must be 1 (open chain)"); return CDZ_EINVAL; }
  // position blocks: greedy runs of bond positions 0..n holding at most CDZ_TB bonds; the bond index space is padded so
  // that block b owns exactly [b*CDZ_TB, (b+1)*CDZ_TB); padding rows / columns stay zero
  tt->off.assign(n + 2, 0);
  tt->posblk.assign(n + 1, 0);
  tt->blk_start.clear();
  tt->blk_start.push_back(0);
  int cur = 0, blk = 0;
  for (int i = 0; i <= n; ++i) {
    if (cur + tt->sigma[i] > CDZ_TB) { ++blk; cur = 0; tt->blk_start.push_back(i); }
    tt->off[i] = blk * CDZ_TB + cur;
    tt->posblk[i] = blk;
    cur += tt->sigma[i];
  }
  tt->NB = blk + 1;
  tt->blk_start.push_back(n + 1);
  tt->S = tt->NB * CDZ_TB;
  tt->off[n + 1] = tt->S;
  // state lists: L_i = distinct (a, b) sorted lexicographically, R_j = distinct (b, c) sorted by (b, c)
  tt->loff.assign(n + 1, 0);
  tt->roff.assign(n + 1, 0);
  tt->op_l.assign(tt->ops.size(), 0);
  tt->op_r.assign(tt->ops.size(), 0);
  tt->ls_a.clear(); tt->ls_x.clear(); tt->rs_y.clear(); tt->rs_c.clear();
  tt->maxL = tt->maxR = tt->maxOps = 1;
  for (int i = 0; i < n; ++i) {
    std::map<int, int> L, R;
    for (int z = tt->opstart[i]; z < tt->opstart[i + 1]; ++z) {
      const cdz_op& o = tt->ops[z];
      L[o.a * 4 + o.b] = 0;
      R[o.b * CDZ_MAX_BOND + o.c] = 0;
    }
    int k = 0;
    for (auto& kv : L) { kv.second = k++; tt->ls_a.push_back(kv.first / 4); tt->ls_x.push_back(kv.first % 4); }
    k = 0;
    for (auto& kv : R) { kv.second = k++; tt->rs_y.push_back(kv.first / CDZ_MAX_BOND); tt->rs_c.push_back(kv.first % CDZ_MAX_BOND); }
    for (int z = tt->opstart[i]; z < tt->opstart[i + 1]; ++z) {
      const cdz_op& o = tt->ops[z];
      tt->op_l[z] = (uint8_t)L[o.a * 4 + o.b];
      tt->op_r[z] = (uint8_t)R[o.b * CDZ_MAX_BOND + o.c];
    }
    tt->loff[i + 1] = tt->loff[i] + (int)L.size();
    tt->roff[i + 1] = tt->roff[i] + (int)R.size();
    tt->maxL = std::max(tt->maxL, (int)L.size());
    tt->maxR = std::max(tt->maxR, (int)R.size());
    tt->maxOps = std::max(tt->maxOps, tt->opstart[i + 1] - tt->opstart[i]);
    if (L.empty()) { cdz_set_error("position without operators"); return CDZ_EINVAL; }
  }
  tt->LS = tt->loff[n];
  tt->RS = tt->roff[n];
  if (tt->maxL > CDZ_MAX_STATES || tt->maxR > CDZ_MAX_STATES) {
    cdz_set_error("more than 16 boundary states at one position");
    return CDZ_EINVAL;
  }
  return CDZ_OK;
}
}  // namespace

// cw_stride = 0: one table codon_logw[64] for every residue; 64: per-position tables codon_logw[L][64]
static int tt_build(const char* aa, int L, int kind, const double* codon_logw, int cw_stride, const double* pair_logw,
                    cdz_tt** out) {
  if (!aa || L <= 0 || !out || (kind != CDZ_TT_SINGLE_CODON && kind != CDZ_TT_CODON_PAIR)) {
    cdz_set_error("cdz_tt_build: bad argument");
    return CDZ_EINVAL;
  }
  if (codon_logw)
    for (size_t c = 0; c < (cw_stride ? (size_t)L * 64 : (size_t)64); ++c)
      if (!std::isfinite(codon_logw[c])) { cdz_set_error("cdz_tt_build: non-finite codon weight"); return CDZ_EINVAL; }
  if (pair_logw)
    for (int c = 0; c < 4096; ++c)
      if (!std::isfinite(pair_logw[c])) { cdz_set_error("cdz_tt_build: non-finite codon-pair weight"); return CDZ_EINVAL; }
  cdz_tt* tt = new (std::nothrow) cdz_tt;
  if (!tt) return CDZ_ENOMEM;
  tt->n = 3 * L;
  tt->kind = kind;
  tt->sigma.assign(tt->n + 1, 1);
  tt->opstart.assign(tt->n + 1, 0);
  std::vector<int> prev;  // codons of the previous residue (pair TT)
  for (int k = 0; k < L; ++k) {
    std::vector<int> cod = codon_set(aa[k]);
    if (cod.empty()) {
      delete tt;
      cdz_set_error(std::string("cdz_tt_build: unknown residue '") + aa[k] + "'");
      return CDZ_EINVAL;
    }
    const int deg = (int)cod.size();
    auto cw = [&](int c) { return codon_logw ? exp(codon_logw[(size_t)k * cw_stride + c]) : 1.0; };
    if (kind == CDZ_TT_SINGLE_CODON) {
      // bonds carry the first base (after 3k) and the third base (after 3k+1), compacted (eq 3.4)
      std::vector<int> firsts, thirds;
      for (int c : cod) { firsts.push_back(c >> 4); thirds.push_back(c & 3); }
      std::map<int, int> rf = rank_map(firsts), rt = rank_map(thirds);
      tt->sigma[3 * k] = 1;
      tt->sigma[3 * k + 1] = (int)rf.size();
      tt->sigma[3 * k + 2] = (int)rt.size();
      tt->opstart[3 * k] = (int)tt->ops.size();
      for (auto& kv : rf) tt->ops.push_back(cdz_op{0, kv.first, kv.second, 1.0});
      tt->opstart[3 * k + 1] = (int)tt->ops.size();
      for (int c : cod) { tt->ops.push_back(cdz_op{rf[c >> 4], (c >> 2) & 3, rt[c & 3], cw(c)}); tt->mid_codon.push_back(c); }
      tt->opstart[3 * k + 2] = (int)tt->ops.size();
      for (auto& kv : rt) tt->ops.push_back(cdz_op{kv.second, kv.first, 0, 1.0});
    } else {
      // bonds carry the codon index; the 5' base holds the codon->codon transition (S3c.ii)
      const int pdeg = k == 0 ? 1 : (int)prev.size();
      tt->sigma[3 * k] = pdeg;
      tt->sigma[3 * k + 1] = deg;
      tt->sigma[3 * k + 2] = deg;
      tt->opstart[3 * k] = (int)tt->ops.size();
      for (int a = 0; a < pdeg; ++a)
        for (int c = 0; c < deg; ++c) {
          double x = (k > 0 && pair_logw) ? exp(pair_logw[prev[a] * 64 + cod[c]]) : 1.0;
          tt->ops.push_back(cdz_op{a, cod[c] >> 4, c, x});
        }
      tt->opstart[3 * k + 1] = (int)tt->ops.size();
      for (int c = 0; c < deg; ++c) { tt->ops.push_back(cdz_op{c, (cod[c] >> 2) & 3, c, cw(cod[c])}); tt->mid_codon.push_back(cod[c]); }
      tt->opstart[3 * k + 2] = (int)tt->ops.size();
      for (int c = 0; c < deg; ++c) tt->ops.push_back(cdz_op{c, cod[c] & 3, c, 1.0});
      prev = cod;
    }
  }
  tt->opstart[tt->n] = (int)tt->ops.size();
  tt->sigma[tt->n] = kind == CDZ_TT_SINGLE_CODON ? 1 : (int)prev.size();
  int rc = finalize_tt(tt);
  if (rc != CDZ_OK) { delete tt; return rc; }
  *out = tt;
  return CDZ_OK;
}

int cdz_codons_of(char aa, int* out) {
  const std::vector<int> v = codon_set(aa);
  for (size_t k = 0; k < v.size(); ++k) out[k] = v[k];
  return (int)v.size();
}

extern "C" int cdz_tt_build(const char* aa, int L, int kind, const double* codon_logw, const double* pair_logw,
                            cdz_tt** out) {
  return tt_build(aa, L, kind, codon_logw, 0, pair_logw, out);
}
extern "C" int cdz_tt_build_pos(const char* aa, int L, int kind, const double* codon_logw_pos, const double* pair_logw,
                                cdz_tt** out) {
  return tt_build(aa, L, kind, codon_logw_pos, 64, pair_logw, out);
}

extern "C" int cdz_tt_from_operators(int n, const int32_t* counts, const cdz_op* ops, cdz_tt** out) {
  if (n <= 0 || !counts || !ops || !out) { cdz_set_error("cdz_tt_from_operators: bad argument"); return CDZ_EINVAL; }
  cdz_tt* tt = new (std::nothrow) cdz_tt;
  if (!tt) return CDZ_ENOMEM;
  tt->n = n;
  tt->sigma.assign(n + 1, 1);
  tt->opstart.assign(n + 1, 0);
  int tot = 0;
  for (int i = 0; i < n; ++i) {
    if (counts[i] <= 0) { delete tt; cdz_set_error("cdz_tt_from_operators: empty operator list"); return CDZ_EINVAL; }
    tt->opstart[i] = tot;
    tot += counts[i];
  }
  tt->opstart[n] = tot;
  tt->ops.assign(ops, ops + tot);
  for (int i = 0; i < n; ++i)
    for (int z = tt->opstart[i]; z < tt->opstart[i + 1]; ++z) {
      const cdz_op& o = tt->ops[z];
      if (o.a < 0 || o.c < 0 || o.b < 0 || o.b > 3 || !(o.x > 0) || !std::isfinite(o.x)) {
        delete tt;
        cdz_set_error("cdz_tt_from_operators: operator out of range (need a,c>=0, b in 0..3, x>0)");
        return CDZ_EINVAL;
      }
      tt->sigma[i] = std::max(tt->sigma[i], o.a + 1);
      tt->sigma[i + 1] = std::max(tt->sigma[i + 1], o.c + 1);
    }
  int rc = finalize_tt(tt);
  if (rc != CDZ_OK) { delete tt; return rc; }
  *out = tt;
  return CDZ_OK;
}

extern "C" void cdz_tt_destroy(cdz_tt* tt) { delete tt; }
extern "C" int cdz_tt_length(const cdz_tt* tt) { return tt ? tt->n : CDZ_EINVAL; }
extern "C" int cdz_tt_describe(const cdz_tt* tt, int32_t* sigma, int32_t* counts) {
  if (!tt) return CDZ_EINVAL;
  if (sigma) for (int i = 0; i <= tt->n; ++i) sigma[i] = tt->sigma[i];
  if (counts) for (int i = 0; i < tt->n; ++i) counts[i] = tt->opstart[i + 1] - tt->opstart[i];
  return (int)tt->ops.size();
}

// ------------------------------------------------------------------------------------------------
// workspace layout
// ------------------------------------------------------------------------------------------------
namespace {
struct Carver {
  char* base;
  size_t used = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <typename T>
  T* take(size_t count) {
    used = (used + 255) & ~size_t(255);
    T* p = base ? (T*)(base + used) : nullptr;
    used += count * sizeof(T);
    return p;
  }
};

// carve every device array; with base == nullptr only sizes are computed
size_t carve(const cdz_tt* tt, void* base, Ctx* c, Ctx** d_ctx) {
  Carver k(base);
  const size_t n = tt->n, S = tt->S, LS = tt->LS, RS = tt->RS, MS = tt->MS, nops = tt->ops.size();
  Ctx tmp;
  Ctx& x = c ? *c : tmp;
  DevTT& t = x.tt;
  t.n = (int)n; t.S = (int)S; t.LS = (int)LS; t.RS = (int)RS; t.MS = (int)MS; t.maxL = tt->maxL; t.maxR = tt->maxR;
  t.NB = tt->NB;
  Ctx* dc = k.take<Ctx>(1);
  if (d_ctx) *d_ctx = dc;
  x.batch = k.take<Ctx>(CDZ_MAX_BATCH);  // device copy of the handles of a batched launch (used on the first handle of the batch)
  t.sig = k.take<int>(n + 1);
  t.off = k.take<int>(n + 2);
  t.opstart = k.take<int>(n + 1);
  t.op_a = k.take<uint8_t>(nops); t.op_b = k.take<uint8_t>(nops); t.op_c = k.take<uint8_t>(nops);
  t.op_l = k.take<uint8_t>(nops); t.op_r = k.take<uint8_t>(nops);
  t.op_codon = k.take<int8_t>(nops);
  t.op_x = k.take<double>(nops);
  t.op_x0 = k.take<double>(nops);
  t.blk_start = k.take<int>(tt->NB + 1);
  t.posblk = k.take<int>(n + 1);
  t.Tbar0 = k.take<double>(n * MS * MS);
  t.loff = k.take<int>(n + 1);
  t.roff = k.take<int>(n + 1);
  t.ls_a = k.take<uint8_t>(LS); t.ls_x = k.take<uint8_t>(LS);
  t.rs_y = k.take<uint8_t>(RS); t.rs_c = k.take<uint8_t>(RS);
  t.lsidx = k.take<int8_t>(n * MS * 4);
  t.rsidx = k.take<int8_t>(n * 4 * MS);
  t.bondpos = k.take<int>(S + 1);
  t.lspos = k.take<int>(LS);
  t.rspos = k.take<int>(RS);
  t.Tbar = k.take<double>(n * MS * MS);
  t.wh = k.take<double>(n + 1);
  DevTab& b = x.tab;
  b.scale = k.take<int>(n + 2);
  b.dP = k.take<int>(n + 2);
  b.EB = k.take<int>(S);
  b.EL = k.take<int>(LS);
  b.ER = k.take<int>(RS);
  b.R = k.take<double>(S);
  {
    // worst case over every batch size the design may be launched in: cdz_nsplit(.., D, B) <= min(CDZ_MAX_SPLIT, D - 1)
    size_t tiles = 1;
    for (int D = 2; D < tt->NB; ++D) tiles = std::max(tiles, (size_t)(tt->NB - D) * (size_t)std::min(CDZ_MAX_SPLIT, D - 1));
    b.GP = k.take<double>(tiles * CDZ_TB * CDZ_TB);
  }
  b.eA = k.take<int>(S);
  b.eB = k.take<int>(S);
  b.ctrl = k.take<int>(64);
  b.result = k.take<double>(16);
  b.Qext = k.take<double>(S);
  b.QB = k.take<double>(LS * RS);
  b.DD = k.take<double>(LS * RS);
  b.D1 = k.take<double>(LS * S);
  b.D2T = k.take<double>(RS * S);
  b.GI = k.take<double>(S * S);
  b.QBS = k.take<double>(S * S);
  b.QM = k.take<double>(S * S);
  b.QM1T = k.take<double>(S * S);
  b.QML = k.take<double>(S * S);
  b.M2 = k.take<double>(S * S);
  b.EM = k.take<double>(S * S);
  b.EMT = k.take<double>(S * S);
  b.QBST = k.take<double>(S * S);
  b.XE = k.take<double>(S * S);
  b.XS = k.take<double>(n * 27 * MS * MS);
  x.cm = k.take<CModel>(1);
  return (k.used + 255) & ~size_t(255);
}
}  // namespace

extern "C" int cdz_workspace_bytes(const cdz_tt* tt, int precision, size_t* bytes) {
  if (!tt || !bytes) { cdz_set_error("cdz_workspace_bytes: null argument"); return CDZ_EINVAL; }
  if (precision != CDZ_FP64 && precision != CDZ_FP32_SCALED) { cdz_set_error("unknown precision"); return CDZ_EINVAL; }
  *bytes = carve(tt, nullptr, nullptr, nullptr);
  return CDZ_OK;
}

static int upload(cdz_tables* T) {
  const cdz_tt* tt = T->tt;
  const cdz_model* m = T->model;
  cudaStream_t st = T->stream;
  const int n = tt->n;
  const DevTT& t = T->h.tt;
  auto up = [&](const void* dst, const void* src, size_t bytes) {
    return cudaMemcpyAsync((void*)dst, src, bytes, cudaMemcpyHostToDevice, st);
  };
  std::vector<uint8_t> oa, ob, oc;
  std::vector<double> ox;
  for (const cdz_op& o : tt->ops) { oa.push_back(o.a); ob.push_back(o.b); oc.push_back(o.c); ox.push_back(o.x); }
  std::vector<int8_t> ocod(tt->ops.size(), -1);
  if (tt->kind >= 0 && !tt->mid_codon.empty()) {
    size_t k = 0;
    for (int r = 0; 3 * r + 1 < n; ++r)
      for (int z = tt->opstart[3 * r + 1]; z < tt->opstart[3 * r + 2]; ++z) ocod[z] = (int8_t)tt->mid_codon[k++];
  }
  // padding bond indices map to the first position of the next block (their table entries are zero)
  std::vector<int> bondpos(tt->S + 1, n), lspos(tt->LS), rspos(tt->RS);
  for (int kb = 0; kb < tt->S; ++kb) bondpos[kb] = std::min(n, tt->blk_start[kb / CDZ_TB + 1]);
  for (int i = 0; i <= n; ++i)
    for (int a = 0; a < tt->sigma[i]; ++a) bondpos[tt->off[i] + a] = i;
  for (int i = 0; i < n; ++i) {
    for (int l = tt->loff[i]; l < tt->loff[i + 1]; ++l) lspos[l] = i;
    for (int r = tt->roff[i]; r < tt->roff[i + 1]; ++r) rspos[r] = i;
  }
  const int MS = tt->MS;
  std::vector<int8_t> lsidx((size_t)n * MS * 4, -1), rsidx((size_t)n * 4 * MS, -1);
  for (int i = 0; i < n; ++i) {
    for (int l = tt->loff[i]; l < tt->loff[i + 1]; ++l) lsidx[((size_t)i * MS + tt->ls_a[l]) * 4 + tt->ls_x[l]] = (int8_t)(l - tt->loff[i]);
    for (int r = tt->roff[i]; r < tt->roff[i + 1]; ++r) rsidx[((size_t)i * 4 + tt->rs_y[r]) * MS + tt->rs_c[r]] = (int8_t)(r - tt->roff[i]);
  }
  std::vector<double> tbar((size_t)n * MS * MS, 0.0);
  for (int i = 0; i < n; ++i)
    for (int z = tt->opstart[i]; z < tt->opstart[i + 1]; ++z)
      tbar[((size_t)i * MS + tt->ops[z].a) * MS + tt->ops[z].c] += tt->ops[z].x;
  std::vector<double> wh(n + 1, 0.0);
  for (int l = m->p.min_hairpin; l <= n; ++l)
    wh[l] = exp(-(m->p.hairpin_a + m->p.hairpin_b * m->kT * log((double)l / m->p.hairpin_l0)) / m->kT);
  CDZ_CUDA(up(t.sig, tt->sigma.data(), sizeof(int) * (n + 1)));
  CDZ_CUDA(up(t.off, tt->off.data(), sizeof(int) * (n + 2)));
  CDZ_CUDA(up(t.opstart, tt->opstart.data(), sizeof(int) * (n + 1)));
  CDZ_CUDA(up(t.op_a, oa.data(), oa.size()));
  CDZ_CUDA(up(t.op_b, ob.data(), ob.size()));
  CDZ_CUDA(up(t.op_c, oc.data(), oc.size()));
  CDZ_CUDA(up(t.op_l, tt->op_l.data(), oa.size()));
  CDZ_CUDA(up(t.op_r, tt->op_r.data(), oa.size()));
  CDZ_CUDA(up(t.op_codon, ocod.data(), ocod.size()));
  CDZ_CUDA(up(t.op_x, ox.data(), sizeof(double) * ox.size()));
  CDZ_CUDA(up(t.op_x0, ox.data(), sizeof(double) * ox.size()));
  CDZ_CUDA(up(t.blk_start, tt->blk_start.data(), sizeof(int) * (tt->NB + 1)));
  CDZ_CUDA(up(t.posblk, tt->posblk.data(), sizeof(int) * (n + 1)));
  CDZ_CUDA(up(t.loff, tt->loff.data(), sizeof(int) * (n + 1)));
  CDZ_CUDA(up(t.roff, tt->roff.data(), sizeof(int) * (n + 1)));
  CDZ_CUDA(up(t.ls_a, tt->ls_a.data(), tt->LS));
  CDZ_CUDA(up(t.ls_x, tt->ls_x.data(), tt->LS));
  CDZ_CUDA(up(t.rs_y, tt->rs_y.data(), tt->RS));
  CDZ_CUDA(up(t.rs_c, tt->rs_c.data(), tt->RS));
  CDZ_CUDA(up(t.lsidx, lsidx.data(), lsidx.size()));
  CDZ_CUDA(up(t.rsidx, rsidx.data(), rsidx.size()));
  CDZ_CUDA(up(t.bondpos, bondpos.data(), sizeof(int) * (tt->S + 1)));
  CDZ_CUDA(up(t.lspos, lspos.data(), sizeof(int) * tt->LS));
  CDZ_CUDA(up(t.rspos, rspos.data(), sizeof(int) * tt->RS));
  CDZ_CUDA(up(t.Tbar, tbar.data(), sizeof(double) * tbar.size()));
  CDZ_CUDA(up(t.Tbar0, tbar.data(), sizeof(double) * tbar.size()));
  CDZ_CUDA(up(t.wh, wh.data(), sizeof(double) * (n + 1)));
  CDZ_CUDA(up(T->h.cm, &m->c, sizeof(CModel)));
  CDZ_CUDA(up(T->d_ctx, &T->h, sizeof(Ctx)));
  CDZ_CUDA(cudaStreamSynchronize(st));  // host staging vectors die at return
  return CDZ_OK;
}

static int make_tables(const cdz_model* m, const cdz_tt* tt, int precision, void* ws, size_t ws_bytes,
                       cudaStream_t st, cdz_tables** out) {
  if (!m || !tt || !out) { cdz_set_error("cdz_inside: null argument"); return CDZ_EINVAL; }
  if (precision != CDZ_FP64 && precision != CDZ_FP32_SCALED) { cdz_set_error("unknown precision"); return CDZ_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cdz_set_error("no CUDA device: this library has no CPU fallback");
    return CDZ_ECUDA;
  }
  cdz_tables* T = new (std::nothrow) cdz_tables;
  if (!T) return CDZ_ENOMEM;
  T->model = m; T->tt = tt; T->precision = precision; T->stream = st;
  size_t need = carve(tt, nullptr, nullptr, nullptr);
  T->bytes = need;
  if (ws) {
    if (ws_bytes < need) { delete T; cdz_set_error("workspace too small"); return CDZ_ENOMEM; }
    T->base = ws;
  } else {
    if (cudaMalloc(&T->base, need) != cudaSuccess) {
      delete T;
      cdz_set_error("cudaMalloc of the DP tables failed");
      return CDZ_ENOMEM;
    }
    T->owns_base = true;
  }
  carve(tt, T->base, &T->h, &T->d_ctx);
  // padding rows / columns of the packed tables are never written by the kernels and must read as zero
  if (cudaMemsetAsync(T->base, 0, need, st) != cudaSuccess) {
    cdz_set_error("cudaMemsetAsync of the DP tables failed");
    cdz_tables_destroy(T);
    return CDZ_ECUDA;
  }
  cudaEventCreate(&T->ev0);
  cudaEventCreate(&T->ev1);
  int rc = upload(T);
  if (rc != CDZ_OK) { cdz_tables_destroy(T); return rc; }
  *out = T;
  return CDZ_OK;
}

int cdz_make_tables(const cdz_model* m, const cdz_tt* tt, int precision, void* ws, size_t ws_bytes, cudaStream_t st, cdz_tables** out) {
  return make_tables(m, tt, precision, ws, ws_bytes, st, out);
}

extern "C" void cdz_tables_destroy(cdz_tables* t) {
  if (!t) return;
  if (t->owns_base && t->base) cudaFree(t->base);
  if (t->ev0) cudaEventDestroy(t->ev0);
  if (t->ev1) cudaEventDestroy(t->ev1);
  for (cudaEvent_t e : t->evs) cudaEventDestroy(e);
  delete t;
}

extern "C" int cdz_tables_logz(cdz_tables* t, double* logZ) {
  if (!t || !logZ) { cdz_set_error("cdz_tables_logz: null argument"); return CDZ_EINVAL; }
  if (!t->done) { cdz_set_error("inside pass has not been launched"); return CDZ_ESTATE; }
  double res[4];
  int ctrl[4];
  CDZ_CUDA(cudaMemcpyAsync(res, t->h.tab.result, sizeof(res), cudaMemcpyDeviceToHost, t->stream));
  CDZ_CUDA(cudaMemcpyAsync(ctrl, t->h.tab.ctrl, sizeof(ctrl), cudaMemcpyDeviceToHost, t->stream));
  CDZ_CUDA(cudaStreamSynchronize(t->stream));
  t->n_rescales = ctrl[0];
  if (ctrl[1] != 0 || !std::isfinite(res[0])) {
    cdz_set_error("dynamic range exceeded (overflow / underflow sentinel)");
    return CDZ_EOVERFLOW;
  }
  *logZ = res[0];
  float ms = 0;
  if (cudaEventElapsedTime(&ms, t->ev0, t->ev1) == cudaSuccess) t->inside_ms = ms;
  return CDZ_OK;
}

extern "C" int cdz_inside_rerun_batch(cdz_tables* const* ts, int B, void* stream) {
  if (!ts || B <= 0) { cdz_set_error("cdz_inside_rerun_batch: bad argument"); return CDZ_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  for (int b = 0; b < B; ++b) {
    if (!ts[b]) { cdz_set_error("null table handle"); return CDZ_EINVAL; }
    ts[b]->stream = st;
  }
  CDZ_CUDA(cudaEventRecord(ts[0]->ev0, st));
  int rc = cdz_launch_inside(ts, B, st);
  if (rc != CDZ_OK) return rc;
  for (int b = 0; b < B; ++b) {
    if (b > 0) cudaEventRecord(ts[b]->ev0, st);
    CDZ_CUDA(cudaEventRecord(ts[b]->ev1, st));
    ts[b]->done = true;
  }
  return CDZ_OK;
}
extern "C" int cdz_inside_rerun(cdz_tables* t, void* stream) { return cdz_inside_rerun_batch(&t, 1, stream); }

extern "C" int cdz_inside_batch(const cdz_model* m, const cdz_tt* const* tts, int B, int precision,
                                void* const* ws, const size_t* ws_bytes, void* stream, cdz_tables** out,
                                double* logZ) {
  if (!tts || !out || B <= 0) { cdz_set_error("cdz_inside_batch: bad argument"); return CDZ_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  for (int b = 0; b < B; ++b) out[b] = nullptr;
  for (int b = 0; b < B; ++b) {
    int rc = make_tables(m, tts[b], precision, ws ? ws[b] : nullptr, ws_bytes ? ws_bytes[b] : 0, st, &out[b]);
    if (rc != CDZ_OK) {
      for (int k = 0; k < b; ++k) { cdz_tables_destroy(out[k]); out[k] = nullptr; }
      return rc;
    }
  }
  int rc = cdz_inside_rerun_batch(out, B, stream);
  if (rc == CDZ_OK && logZ)
    for (int b = 0; b < B && rc == CDZ_OK; ++b) rc = cdz_tables_logz(out[b], &logZ[b]);
  if (rc != CDZ_OK)
    for (int b = 0; b < B; ++b) { cdz_tables_destroy(out[b]); out[b] = nullptr; }
  return rc;
}

extern "C" int cdz_inside(const cdz_model* m, const cdz_tt* tt, int precision, void* ws, size_t ws_bytes,
                          void* stream, cdz_tables** out, double* logZ) {
  void* wsv[1] = {ws};
  size_t wsb[1] = {ws_bytes};
  return cdz_inside_batch(m, &tt, 1, precision, wsv, wsb, stream, out, logZ);
}

extern "C" int cdz_tables_info(cdz_tables* t, cdz_info* info) {
  if (!t || !info) { cdz_set_error("cdz_tables_info: null argument"); return CDZ_EINVAL; }
  const cdz_tt* tt = t->tt;
  memset(info, 0, sizeof(*info));
  const int n = tt->n;
  info->n = n;
  info->sigma_bar = tt->sigma_bar;
  info->n_left_states = tt->LS;
  info->n_right_states = tt->RS;
  info->precision = t->precision;
  info->n_rescales = t->n_rescales;
  // N_cc = sum_d (n-d) max(0, d-8); N_loop = #(i,j,l1,l2), l1+l2<=max_interior, inner span >= 5 nt
  const int mh = t->model->p.min_hairpin, mi = t->model->p.max_interior;
  double ncc = 0, nloop = 0;
  for (int d = 0; d < n; ++d) {
    ncc += (double)(n - d) * std::max(0, d - 2 * (mh + 1));
    int cnt = 0;
    for (int l1 = 0; l1 <= mi; ++l1)
      for (int l2 = 0; l1 + l2 <= mi; ++l2)
        if (d - 2 - l1 - l2 >= mh + 1) ++cnt;
    nloop += (double)(n - d) * cnt;
  }
  info->n_cc = ncc;
  info->n_loop = nloop;
  // exact split MACs: sum over (i<k<=j) of Sigma_i Sigma_k Sigma_{j+1} = sum_k (prefix_i)(suffix_j)
  double mac = 0, pre = 0;
  std::vector<double> suf(n + 2, 0.0);
  for (int j = n - 1; j >= 0; --j) suf[j] = suf[j + 1] + tt->sigma[j + 1];
  for (int k = 1; k < n; ++k) {
    pre += tt->sigma[k - 1];
    mac += pre * tt->sigma[k] * suf[k];
  }
  info->split_mac = mac;
  info->table_bytes = (double)t->bytes;
  info->bytes_per_cell = (double)t->bytes / (0.5 * n * (n + 1.0));
  double sc = 0;
  if (t->done) {
    double res[4];
    if (cudaMemcpy(res, t->h.tab.result, sizeof(res), cudaMemcpyDeviceToHost) == cudaSuccess) sc = res[2];
    float ms = 0;
    if (cudaEventElapsedTime(&ms, t->ev0, t->ev1) == cudaSuccess) t->inside_ms = ms;
  }
  info->log_scale = sc;
  info->inside_ms = t->inside_ms;
  return CDZ_OK;
}

extern "C" int cdz_set_profiling(cdz_tables* t, int on) {
  if (!t) { cdz_set_error("cdz_set_profiling: null handle"); return CDZ_EINVAL; }
  t->profile = on != 0;
  return CDZ_OK;
}

extern "C" int cdz_profile(cdz_tables* t, double* ms_out, int64_t* launches_out) {
  if (!t) { cdz_set_error("cdz_profile: null handle"); return CDZ_EINVAL; }
  if (!t->done) { cdz_set_error("inside pass has not been launched"); return CDZ_ESTATE; }
  CDZ_CUDA(cudaStreamSynchronize(t->stream));
  if (ms_out) {
    for (int k = 0; k < CDZ_NCLASS; ++k) ms_out[k] = 0.0;
    for (size_t k = 0; k + 1 < t->ev_class.size() && k + 1 < t->evs.size(); ++k) {
      float ms = 0;
      if (t->ev_class[k] >= 0 && cudaEventElapsedTime(&ms, t->evs[k], t->evs[k + 1]) == cudaSuccess)
        ms_out[t->ev_class[k]] += ms;
    }
  }
  if (launches_out)
    for (int k = 0; k < CDZ_NCLASS; ++k) launches_out[k] = t->launches[k];
  return CDZ_OK;
}

extern "C" int cdz_debug_set_rescale_start(cdz_tables* t, int first) {
  if (!t || first < 1) { cdz_set_error("cdz_debug_set_rescale_start: bad argument"); return CDZ_EINVAL; }
  t->rescale_first = first;
  return CDZ_OK;
}

// debug / parity access ------------------------------------------------------------------------------
extern "C" int cdz_tables_cell(cdz_tables* t, int which, int i, int j, double* out, int* shift_out) {
  if (!t || !out || i < 0 || j < i || j >= t->tt->n || which < 0 || which > 5) {
    cdz_set_error("cdz_tables_cell: bad argument");
    return CDZ_EINVAL;
  }
  if (!t->done) { cdz_set_error("inside pass has not been launched"); return CDZ_ESTATE; }
  const cdz_tt* tt = t->tt;
  CDZ_CUDA(cudaStreamSynchronize(t->stream));
  const int Si = tt->sigma[i], Sj = tt->sigma[j + 1], S = tt->S;
  std::vector<int> P(tt->n + 2);
  CDZ_CUDA(cudaMemcpy(P.data(), t->h.tab.scale, sizeof(int) * (tt->n + 1), cudaMemcpyDeviceToHost));
  if (shift_out) *shift_out = P[j + 1] - P[i];
  auto rd = [&](const double* p) { double v = 0; cudaMemcpy(&v, p, sizeof(double), cudaMemcpyDeviceToHost); return v; };
  if (which == 0) {
    for (int k = 0; k < Si * 16 * Sj; ++k) out[k] = 0;
    const int nl = tt->loff[i + 1] - tt->loff[i], nr = tt->roff[j + 1] - tt->roff[j];
    for (int l = 0; l < nl; ++l)
      for (int r = 0; r < nr; ++r) {
        int a = tt->ls_a[tt->loff[i] + l], x = tt->ls_x[tt->loff[i] + l];
        int y = tt->rs_y[tt->roff[j] + r], c = tt->rs_c[tt->roff[j] + r];
        out[((a * 4 + x) * 4 + y) * Sj + c] = rd(t->h.tab.QB + (size_t)(tt->loff[i] + l) * tt->RS + tt->roff[j] + r);
      }
    return Si * 16 * Sj;
  }
  const double* tabs[6] = {nullptr, t->h.tab.QBS, t->h.tab.QM1T, t->h.tab.QML, t->h.tab.M2, t->h.tab.QM};
  for (int a = 0; a < Si; ++a)
    for (int c = 0; c < Sj; ++c) {
      size_t r = tt->off[i] + a, q = tt->off[j + 1] + c;
      out[a * Sj + c] = rd(tabs[which] + (which == 2 ? q * S + r : r * S + q));
    }
  return Si * Sj;
}

extern "C" int cdz_tables_logqext(cdz_tables* t, int j, int c, double* out) {
  if (!t || !out || j < -1 || j >= t->tt->n || c < 0 || c >= t->tt->sigma[j + 1]) {
    cdz_set_error("cdz_tables_logqext: bad argument");
    return CDZ_EINVAL;
  }
  if (!t->done) { cdz_set_error("inside pass has not been launched"); return CDZ_ESTATE; }
  CDZ_CUDA(cudaStreamSynchronize(t->stream));
  double v = 0;
  int P = 0;
  CDZ_CUDA(cudaMemcpy(&v, t->h.tab.Qext + (size_t)t->tt->off[j + 1] + c, sizeof(double), cudaMemcpyDeviceToHost));
  CDZ_CUDA(cudaMemcpy(&P, t->h.tab.scale + (j + 1), sizeof(int), cudaMemcpyDeviceToHost));
  *out = log(v) + P * 0.6931471805599453;
  return CDZ_OK;
}

// Work on `st` that reads the tables must run after the inside pass, which may have been launched on another stream.
int cdz_wait_pass(cdz_tables* t, cudaStream_t st) {
  if (st != t->stream) CDZ_CUDA(cudaStreamWaitEvent(st, t->ev1, 0));
  return CDZ_OK;
}

extern "C" int cdz_sample(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_dev, int32_t* pair_dev, void* stream) {
  if (!t || J < 0 || !seq_dev || !pair_dev) { cdz_set_error("cdz_sample: bad argument"); return CDZ_EINVAL; }
  if (!t->done) { cdz_set_error("cdz_sample before cdz_inside"); return CDZ_ESTATE; }
  if (J == 0) return CDZ_OK;
  const int rc = cdz_wait_pass(t, (cudaStream_t)stream);
  if (rc != CDZ_OK) return rc;
  return cdz_launch_sample(t, J, seed, seq_dev, pair_dev, (cudaStream_t)stream);
}

extern "C" int cdz_marginals_workspace_bytes(const cdz_tables* t, size_t* bytes) {
  if (!t || !bytes) { cdz_set_error("cdz_marginals_workspace_bytes: null argument"); return CDZ_EINVAL; }
  *bytes = cdz_outside_carve(t->tt, nullptr, nullptr);
  return CDZ_OK;
}

extern "C" int cdz_marginals(cdz_tables* t, void* workspace_dev, size_t workspace_bytes, double* bpp_dev, double* base_dev,
                             double* codon_dev, void* stream) {
  if (!t) { cdz_set_error("cdz_marginals: null handle"); return CDZ_EINVAL; }
  if (!t->done) { cdz_set_error("cdz_marginals before cdz_inside"); return CDZ_ESTATE; }
  if (!bpp_dev && !base_dev && !codon_dev) return CDZ_OK;
  if (codon_dev && (t->tt->kind < 0 || t->tt->mid_codon.empty())) {
    cdz_set_error("cdz_marginals: codon marginals need a tensor train made by cdz_tt_build (generic operator lists carry no codon labels)");
    return CDZ_EINVAL;
  }
  if (t->tt->maxOps > 256) { cdz_set_error("cdz_marginals: more than 256 operators at one position"); return CDZ_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  int rc = cdz_wait_pass(t, st);
  if (rc != CDZ_OK) return rc;
  const size_t need = cdz_outside_carve(t->tt, nullptr, nullptr);
  void* ws = workspace_dev;
  if (ws) {
    if (workspace_bytes < need) { cdz_set_error("cdz_marginals: workspace too small (cdz_marginals_workspace_bytes)"); return CDZ_ENOMEM; }
  } else if (cudaMallocAsync(&ws, need, st) != cudaSuccess) {  // stream-ordered: no synchronisation
    cudaGetLastError();
    cdz_set_error("cdz_marginals: out of device memory for the adjoint tables");
    return CDZ_ENOMEM;
  }
  Adj A;
  cdz_outside_carve(t->tt, ws, &A);
  A.status = t->h.tab.ctrl + 8;  // lives in the tables' own workspace: readable after a library-owned workspace has been freed
  CDZ_CUDA(cudaMemsetAsync(A.status, 0, sizeof(int), st));
  rc = cdz_launch_outside(t, A, need, bpp_dev, base_dev, codon_dev, st);
  if (!workspace_dev) cudaFreeAsync(ws, st);
  t->marg_stream = st;
  return rc;
}

extern "C" int cdz_marginals_status(cdz_tables* t) {
  if (!t) { cdz_set_error("cdz_marginals_status: null handle"); return CDZ_EINVAL; }
  int flag = 0;
  CDZ_CUDA(cudaMemcpyAsync(&flag, t->h.tab.ctrl + 8, sizeof(int), cudaMemcpyDeviceToHost, t->marg_stream));
  CDZ_CUDA(cudaStreamSynchronize(t->marg_stream));
  if (flag != 0) {
    cdz_set_error("cdz_marginals: an operator usage left [0,1] or the usages of a position do not sum to 1 (dynamic range exceeded)");
    return CDZ_EOVERFLOW;
  }
  return CDZ_OK;
}

extern "C" int cdz_run_host(cdz_tables* t, int J, uint64_t seed, uint8_t* seq_host, int32_t* pair_host,
                            double* logZ_host, void* stream) {
  if (!t) { cdz_set_error("cdz_run_host: null handle"); return CDZ_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  // host -> device: the design's operator weights are re-uploaded (inputs of the step)
  int rc = CDZ_OK;
  {
    // re-upload of the tensor train (h2d of the step's inputs)
    extern int cdz_reupload(cdz_tables*);
    rc = cdz_reupload(t);
    if (rc != CDZ_OK) return rc;
  }
  rc = cdz_inside_rerun(t, stream);
  if (rc != CDZ_OK) return rc;
  const size_t n = t->tt->n;
  uint8_t* sd = nullptr;
  int32_t* pd = nullptr;
  if (J > 0) {
    CDZ_CUDA(cudaMallocAsync((void**)&sd, (size_t)J * n, st));
    CDZ_CUDA(cudaMallocAsync((void**)&pd, (size_t)J * n * sizeof(int32_t), st));
    rc = cdz_launch_sample(t, J, seed, sd, pd, st);
    if (rc != CDZ_OK) return rc;
    if (seq_host) CDZ_CUDA(cudaMemcpyAsync(seq_host, sd, (size_t)J * n, cudaMemcpyDeviceToHost, st));
    if (pair_host) CDZ_CUDA(cudaMemcpyAsync(pair_host, pd, (size_t)J * n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CDZ_CUDA(cudaFreeAsync(sd, st));
    CDZ_CUDA(cudaFreeAsync(pd, st));
  }
  double lz = 0;
  rc = cdz_tables_logz(t, &lz);
  if (logZ_host) *logZ_host = lz;
  return rc;
}

int cdz_reupload(cdz_tables* t) { return upload(t); }
