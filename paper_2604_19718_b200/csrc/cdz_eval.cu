// cdz_eval.cu -- batched fixed-sequence evaluation of sampled sequences (PAPER.md S4f line 779: "q(phi) and P^phi for
// the samples ... more expensive than computing q_psi and the samples ... embarrassingly parallelizable").
//
// A fixed sequence phi is the tensor train with ONE operator (0, phi_i, 0, 1) per position (operator format of PAPER.md lines 545-557), so
// its partition function log Z(phi) -- ordinary McCaskill under the same loop model -- comes out of the same kernels: the J sequences
// are advanced together, chunk by chunk, by cdz_inside_batch; the unpaired probabilities P(i unpaired | phi) come from cdz_marginals.
// log W(phi) = log e_0^T prod_i T_i^{phi_i} 1 (eq 3.1 with the open boundaries of S3c) is evaluated on the host from the design's
// operator lists (O(n) per sequence).  Host orchestration only: every DP step runs in the CUDA kernels.
#include <math.h>

#include <algorithm>
#include <vector>

#include "cdz_internal.h"

extern "C" int cdz_eval_sequences(const cdz_model* m, const cdz_tt* design, int n, int J, const uint8_t* seq_host, int max_batch,
                                  double* logZ_host, double* logW_host, double* unpaired_host, void* stream) {
  if (!m || !seq_host || !logZ_host || n <= 0 || J < 0 || (design && design->n != n)) {
    cdz_set_error("cdz_eval_sequences: bad argument (model, sequences and logZ_host are required; the design must have n positions)");
    return CDZ_EINVAL;
  }
  if (logW_host && !design) { cdz_set_error("cdz_eval_sequences: logW_host needs the design's tensor train"); return CDZ_EINVAL; }
  for (size_t k = 0; k < (size_t)J * n; ++k)
    if (seq_host[k] > 3) { cdz_set_error("cdz_eval_sequences: nucleotide code outside 0..3"); return CDZ_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  // ---- sequence weights from the design's operator lists (host) ----------------------------------------------------------------------
  if (logW_host) {
    std::vector<double> v(CDZ_MAX_BOND), w(CDZ_MAX_BOND);
    for (int s = 0; s < J; ++s) {
      const uint8_t* phi = seq_host + (size_t)s * n;
      std::fill(v.begin(), v.end(), 0.0);
      v[0] = 1.0;
      double lg = 0.0;
      for (int i = 0; i < n; ++i) {
        std::fill(w.begin(), w.end(), 0.0);
        for (int z = design->opstart[i]; z < design->opstart[i + 1]; ++z) {
          const cdz_op& o = design->ops[z];
          if (o.b == phi[i]) w[o.c] += v[o.a] * o.x;
        }
        double mx = 0.0;
        for (double x : w) mx = std::max(mx, x);
        if (!(mx > 0.0)) { lg = -INFINITY; break; }  // phi is not a sequence of the design space
        for (int c = 0; c < CDZ_MAX_BOND; ++c) v[c] = w[c] / mx;
        lg += log(mx);
      }
      if (std::isfinite(lg)) {
        double tot = 0.0;
        for (int c = 0; c < design->sigma[n]; ++c) tot += v[c];
        lg += log(tot);
      }
      logW_host[s] = lg;
    }
  }
  if (J == 0) return CDZ_OK;
  // ---- chunk size from the free device memory -----------------------------------------------------------------------------------------
  std::vector<int32_t> counts(n, 1);
  std::vector<cdz_op> ops(n);
  auto make_tt = [&](const uint8_t* phi, cdz_tt** out) {
    for (int i = 0; i < n; ++i) ops[i] = cdz_op{0, phi[i], 0, 1.0};
    return cdz_tt_from_operators(n, counts.data(), ops.data(), out);
  };
  cdz_tt* probe = nullptr;
  int rc = make_tt(seq_host, &probe);
  if (rc != CDZ_OK) return rc;
  size_t per = 0, fr = 0, total = 0;
  cdz_workspace_bytes(probe, CDZ_FP64, &per);
  cdz_tt_destroy(probe);
  CDZ_CUDA(cudaMemGetInfo(&fr, &total));
  size_t extra = 0;
  if (unpaired_host) extra = (size_t)n * n * sizeof(double);
  const size_t budget = (size_t)(0.8 * (double)fr);
  if (per + extra > budget) { cdz_set_error("cdz_eval_sequences: one fixed-sequence pass does not fit the free device memory"); return CDZ_ENOMEM; }
  int B = (int)std::min<size_t>((budget - extra) / per, (size_t)CDZ_MAX_BATCH);
  if (max_batch > 0) B = std::min(B, max_batch);
  B = std::max(1, std::min(B, J));
  double* bpp = nullptr;
  if (unpaired_host) CDZ_CUDA(cudaMalloc((void**)&bpp, extra));
  // ---- chunks ---------------------------------------------------------------------------------------------------------------------------------
  for (int s0 = 0; s0 < J && rc == CDZ_OK; s0 += B) {
    const int nb = std::min(B, J - s0);
    std::vector<cdz_tt*> tts(nb, nullptr);
    std::vector<cdz_tables*> tabs(nb, nullptr);
    for (int b = 0; b < nb && rc == CDZ_OK; ++b) rc = make_tt(seq_host + (size_t)(s0 + b) * n, &tts[b]);
    if (rc == CDZ_OK) rc = cdz_inside_batch(m, tts.data(), nb, CDZ_FP64, nullptr, nullptr, stream, tabs.data(), logZ_host + s0);
    if (rc == CDZ_OK && unpaired_host)
      for (int b = 0; b < nb && rc == CDZ_OK; ++b) {
        rc = cdz_marginals(tabs[b], nullptr, 0, bpp, nullptr, nullptr, stream);
        if (rc == CDZ_OK) rc = cdz_marginals_status(tabs[b]);
        if (rc == CDZ_OK &&
            cudaMemcpy2DAsync(unpaired_host + (size_t)(s0 + b) * n, sizeof(double), bpp, (size_t)(n + 1) * sizeof(double), sizeof(double),
                              n, cudaMemcpyDeviceToHost, st) != cudaSuccess) {
          cdz_set_error("cdz_eval_sequences: copy of the unpaired probabilities failed");
          rc = CDZ_ECUDA;
        }
        if (rc == CDZ_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = CDZ_ECUDA;
      }
    for (int b = 0; b < nb; ++b) {
      if (tabs[b]) cdz_tables_destroy(tabs[b]);
      if (tts[b]) cdz_tt_destroy(tts[b]);
    }
  }
  if (bpp) cudaFree(bpp);
  return rc;
}
