// cdz_freq.cu -- frequency matching (PAPER.md S4e lines 751-771, Alg S4.6 "MatchFrequencies", Fig 8).
//
// Goal: per-codon multiplicative bonuses f (log f = the codon_logw table of cdz_tt_build) such that the codon frequencies of the design
// distribution, b[c] = sum_k p_k(c) with p_k the exact codon marginals (eq 4.3), equal the target frequencies b*.  As in Alg S4.6 the
// targets are the frequencies of the structure-free uniform distribution U(psi) with bonuses f*:  b*[c] = sum_{k: c codes aa_k}
// f*_c / sum_{c' codes aa_k} f*_c'.  Iteration (prose of S4e, steps 1-3): compute the exact marginals with the current bonuses; stop when
// || log(b / b*) ||_inf < rtol; else multiply f by b* / b ("the ratio of desired frequencies divided by the achieved frequencies"; the
// update line of the printed pseudo-code has the ratio upside down).  Optionally with Anderson acceleration over the
// whole history (line 771: "a standard implementation ... no history size limit").
// Host orchestration of the CUDA path: every iteration is cdz_tt_build + cdz_inside + cdz_marginals (codon marginals) on the device.
#include <math.h>

#include <algorithm>
#include <vector>

#include "cdz_internal.h"

int cdz_codons_of(char aa, int* out);  // cdz_host.cu: sense codons of a residue, ascending; returns the count (0 if unknown)

namespace {
// least squares  min || r - D gamma ||  by modified Gram-Schmidt QR (D: rows x cols, column-major vectors); columns that are
// numerically dependent on the previous ones get gamma = 0
std::vector<double> lstsq(const std::vector<std::vector<double>>& D, const std::vector<double>& r) {
  const size_t cols = D.size(), rows = r.size();
  std::vector<std::vector<double>> Q(cols, std::vector<double>(rows, 0.0));
  std::vector<std::vector<double>> R(cols, std::vector<double>(cols, 0.0));
  std::vector<bool> dead(cols, false);
  for (size_t j = 0; j < cols; ++j) {
    std::vector<double> v = D[j];
    double n0 = 0.0;
    for (double x : v) n0 += x * x;
    for (size_t i = 0; i < j; ++i) {
      if (dead[i]) continue;
      double d = 0.0;
      for (size_t k = 0; k < rows; ++k) d += Q[i][k] * v[k];
      R[i][j] = d;
      for (size_t k = 0; k < rows; ++k) v[k] -= d * Q[i][k];
    }
    double nn = 0.0;
    for (double x : v) nn += x * x;
    if (!(nn > 1e-20 * std::max(n0, 1e-300))) { dead[j] = true; continue; }
    R[j][j] = sqrt(nn);
    for (size_t k = 0; k < rows; ++k) Q[j][k] = v[k] / R[j][j];
  }
  std::vector<double> qtr(cols, 0.0), gamma(cols, 0.0);
  for (size_t j = 0; j < cols; ++j)
    if (!dead[j])
      for (size_t k = 0; k < rows; ++k) qtr[j] += Q[j][k] * r[k];
  for (size_t jj = cols; jj-- > 0;) {
    if (dead[jj]) continue;
    double s = qtr[jj];
    for (size_t i = jj + 1; i < cols; ++i)
      if (!dead[i]) s -= R[jj][i] * gamma[i];
    gamma[jj] = s / R[jj][jj];
  }
  return gamma;
}
}  // namespace

extern "C" int cdz_match_frequencies(const cdz_model* m, const char* aa, int L, int kind, const double* logf_star,
                                     const double* pair_logw, double rtol, int max_iter, int anderson, double* logf_out,
                                     double* err_history, int* n_iter_out, void* stream) {
  if (!m || !aa || L <= 0 || !logf_star || !logf_out || !(rtol > 0) || max_iter <= 0) {
    cdz_set_error("cdz_match_frequencies: bad argument");
    return CDZ_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  // ---- target frequencies b* from U(psi) with the bonuses f* ---------------------------------------------------------------------------
  std::vector<double> bstar(64, 0.0);
  for (int k = 0; k < L; ++k) {
    int cod[8];
    const int deg = cdz_codons_of(aa[k], cod);
    if (deg == 0) { cdz_set_error("cdz_match_frequencies: unknown residue"); return CDZ_EINVAL; }
    double tot = 0.0;
    for (int t = 0; t < deg; ++t) tot += exp(logf_star[cod[t]]);
    for (int t = 0; t < deg; ++t) bstar[cod[t]] += exp(logf_star[cod[t]]) / tot;
  }
  std::vector<int> active;  // codons with a requested frequency > 0 (the others are left alone, line 769)
  for (int c = 0; c < 64; ++c)
    if (bstar[c] > 0.0) active.push_back(c);
  std::vector<double> logf(logf_star, logf_star + 64);
  for (int c = 0; c < 64; ++c)
    if (!std::isfinite(logf[c])) { cdz_set_error("cdz_match_frequencies: non-finite bonus"); return CDZ_EINVAL; }
  // ---- device buffers, reused by every iteration -----------------------------------------------------------------------------------------
  cdz_tt* tt = nullptr;
  int rc = cdz_tt_build(aa, L, kind, logf.data(), pair_logw, &tt);
  if (rc != CDZ_OK) return rc;
  size_t ws_bytes = 0, mw_bytes = 0;
  cdz_workspace_bytes(tt, CDZ_FP64, &ws_bytes);
  void *ws = nullptr, *mws = nullptr;
  double* codon_dev = nullptr;
  std::vector<double> codon((size_t)L * 64);
  auto cleanup = [&]() {
    if (tt) cdz_tt_destroy(tt);
    if (ws) cudaFree(ws);
    if (mws) cudaFree(mws);
    if (codon_dev) cudaFree(codon_dev);
  };
  if (cudaMalloc(&ws, ws_bytes) != cudaSuccess || cudaMalloc((void**)&codon_dev, sizeof(double) * codon.size()) != cudaSuccess) {
    cudaGetLastError();
    cleanup();
    cdz_set_error("cdz_match_frequencies: out of device memory");
    return CDZ_ENOMEM;
  }
  std::vector<std::vector<double>> hist_x, hist_g;  // Anderson history: iterates x_j = log f (active entries) and g(x_j) = x_j + log(b*/b)
  int it = 0;
  for (; it < max_iter; ++it) {
    if (it > 0) {
      cdz_tt_destroy(tt);
      tt = nullptr;
      rc = cdz_tt_build(aa, L, kind, logf.data(), pair_logw, &tt);
      if (rc != CDZ_OK) break;
    }
    cdz_tables* tab = nullptr;
    rc = cdz_inside(m, tt, CDZ_FP64, ws, ws_bytes, stream, &tab, nullptr);
    if (rc != CDZ_OK) break;
    if (!mws) {
      cdz_marginals_workspace_bytes(tab, &mw_bytes);
      if (cudaMalloc(&mws, mw_bytes) != cudaSuccess) {
        cudaGetLastError();
        cdz_tables_destroy(tab);
        cdz_set_error("cdz_match_frequencies: out of device memory for the adjoint tables");
        rc = CDZ_ENOMEM;
        break;
      }
    }
    rc = cdz_marginals(tab, mws, mw_bytes, nullptr, nullptr, codon_dev, stream);
    if (rc == CDZ_OK) rc = cdz_marginals_status(tab);
    if (rc == CDZ_OK && cudaMemcpyAsync(codon.data(), codon_dev, sizeof(double) * codon.size(), cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = CDZ_ECUDA;
    if (rc == CDZ_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = CDZ_ECUDA;
    cdz_tables_destroy(tab);
    if (rc != CDZ_OK) break;
    // b <- accumulated codon frequencies; error = || log(b / b*) ||_inf over the requested codons
    std::vector<double> b(64, 0.0);
    for (int k = 0; k < L; ++k)
      for (int c = 0; c < 64; ++c) b[c] += codon[(size_t)k * 64 + c];
    double err = 0.0;
    std::vector<double> r(active.size());
    for (size_t a = 0; a < active.size(); ++a) {
      r[a] = log(bstar[active[a]] / b[active[a]]);
      err = std::max(err, fabs(r[a]));
    }
    if (err_history) err_history[it] = err;
    if (!(err >= rtol)) { ++it; break; }  // converged (also leaves on NaN)
    // f <- f b*/b, optionally Anderson-accelerated
    std::vector<double> x(active.size()), g(active.size());
    for (size_t a = 0; a < active.size(); ++a) { x[a] = logf[active[a]]; g[a] = x[a] + r[a]; }
    std::vector<double> xn = g;
    if (anderson && !hist_x.empty()) {
      // residuals r_j = g_j - x_j; minimise || r_k - sum_j gamma_j (r_{j+1} - r_j) ||, x_{k+1} = g_k - sum_j gamma_j (g_{j+1} - g_j)
      std::vector<std::vector<double>> X = hist_x, G = hist_g;
      X.push_back(x);
      G.push_back(g);
      const size_t mcols = X.size() - 1;
      std::vector<std::vector<double>> dR(mcols, std::vector<double>(active.size())), dG = dR;
      for (size_t j = 0; j < mcols; ++j)
        for (size_t a = 0; a < active.size(); ++a) {
          dG[j][a] = G[j + 1][a] - G[j][a];
          dR[j][a] = (G[j + 1][a] - X[j + 1][a]) - (G[j][a] - X[j][a]);
        }
      const std::vector<double> gamma = lstsq(dR, r);
      for (size_t j = 0; j < mcols; ++j)
        for (size_t a = 0; a < active.size(); ++a) xn[a] -= gamma[j] * dG[j][a];
    }
    hist_x.push_back(x);
    hist_g.push_back(g);
    for (size_t a = 0; a < active.size(); ++a) logf[active[a]] = xn[a];
  }
  cleanup();
  if (rc != CDZ_OK) return rc;
  for (int c = 0; c < 64; ++c) logf_out[c] = logf[c];
  if (n_iter_out) *n_iter_out = it;
  return CDZ_OK;
}
