// bgo_oracle.cpp -- CPU ORACLE for the combined MoE layer.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.  It shares no code, header, table or helper
// with the CUDA path (paper_2606_21712_b200/csrc); neither includes the other.
//
// What it computes: `h_out <- MoE(h_combined, l)` (Algorithm 1 line 8),
// where h_combined is the concatenation COMBINE produces.  The paper
// does not spell out the MoE arithmetic; it is fixed by BASELINE.json
// `north_star` and restated in SURVEY.md §8(c) / DESIGN.md §"Definition":
//
//   L[t,e]   = sum_j widen(hidden[t,j]) * W_r[j,e] (+ b_r[e])            (a1)
//   sel      = k experts maximal under  a > b  <=>  L[a]>L[b] or (L[a]==L[b] and a<b)   (a2, S3)
//   idx[t,s] = s-th element of sel under that order (s=0 largest)
//   w[t,s]   = exp(L[idx s]-L[idx 0]) / sum_s' exp(L[idx s']-L[idx 0])                  (a2, S2)
//   counts[e]= |{(t,s): idx[t,s]=e}|; offsets = exclusive scan, offsets[E]=T*k          (a3,a4)
//   row_src  = flat indices i=t*k+s sorted by (idx[i], i); inv_perm[row_src[r]] = r     (a5, S8)
//   x_perm[r]= hidden[row_src[r]/k]                                                      (a6)
//   H[r,:]   = silu(x W_gate[e]) (.) (x W_up[e]),  silu(z)=z/(1+exp(-z))                 (a7, S12)
//   Y[r,:]   = H[r,:] W_down[e]                                                          (a8)
//   out[t,:] = sum_{s=0..k-1} w[t,s] * Y[inv_perm[t*k+s],:]                              (a9, S11)
//
// Precision: bf16 inputs are widened exactly; every floating-point step is fp64 with no
// intermediate bf16 rounding; logits and gate weights are rounded once to fp32 (they are
// fp32 artefacts of the interface); `out` stays fp64.  Loops are written in the order the
// definition states (j ascending, slots ascending); there is no blocking or fusion.
// OpenMP only parallelises over independent rows / tokens.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms (one-hot / zero rows),
// numpy stable-sort brute force for top-k and the permutation, counts sum to T*k, bijection,
// gate weights sum to 1 / k=1 => 1.0 / k=E => full softmax, E=1,k=1 => dense SwiGLU FFN via
// numpy fp64 matmul, Y[r,:]=r closed form for un-permute, W_down*2 doubles the output,
// gate<->up swap changes it, per-token brute force == batched path, combine-invariance.
// PARITY UNPINNED: absolute expert-output values on random data beyond those pins -- the
// paper prints no worked numeric example of the MoE layer (last row).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Exact widening of a bf16 bit pattern: bf16 is the upper 16 bits of an IEEE binary32.
inline double widen_bf16(uint16_t b) {
  uint32_t u = static_cast<uint32_t>(b) << 16;
  float f;
  std::memcpy(&f, &u, sizeof f);
  return static_cast<double>(f);
}

// The strict total order of reading S3:  a beats b  <=>  L[a] > L[b] or (L[a] == L[b] and a < b).
// Every comparison with a NaN is false (reading S4), -0.0 == +0.0 is a tie.
inline bool beats(const float* L, int a, int b) {
  return (L[a] > L[b]) || (L[a] == L[b] && a < b);
}

// Top-k of one token by k passes of "best remaining expert" (selection by the definition).
void topk_one(const float* L, int E, int k, int32_t* idx, float* w) {
  std::vector<char> taken(E, 0);
  for (int s = 0; s < k; ++s) {
    int best = -1;
    for (int e = 0; e < E; ++e) {
      if (taken[e]) continue;
      if (best < 0 || beats(L, e, best)) best = e;
    }
    taken[best] = 1;
    idx[s] = best;
  }
  // softmax over the k selected logits with max subtraction (slot 0 holds the max)
  double denom = 0.0;
  std::vector<double> ex(k);
  for (int s = 0; s < k; ++s) {
    ex[s] = std::exp(static_cast<double>(L[idx[s]]) - static_cast<double>(L[idx[0]]));
    denom += ex[s];
  }
  for (int s = 0; s < k; ++s) w[s] = static_cast<float>(ex[s] / denom);
}

inline double silu(double z) { return z / (1.0 + std::exp(-z)); }

// One row through one expert: y[0..d) = (silu(x Wg) (.) (x Wu)) Wd, all fp64.
// Wg, Wu: [d,f] (f contiguous); Wd: [f,d] (d contiguous).  g,u,h: scratch of size f.
void expert_row(const double* x, const uint16_t* Wg, const uint16_t* Wu, const uint16_t* Wd,
                int d, int f, double* g, double* u, double* y) {
  for (int c = 0; c < f; ++c) { g[c] = 0.0; u[c] = 0.0; }
  for (int j = 0; j < d; ++j) {            // j ascending for every output column c
    const double xj = x[j];
    const uint16_t* wg = Wg + static_cast<size_t>(j) * f;
    const uint16_t* wu = Wu + static_cast<size_t>(j) * f;
    for (int c = 0; c < f; ++c) {
      g[c] += xj * widen_bf16(wg[c]);
      u[c] += xj * widen_bf16(wu[c]);
    }
  }
  for (int c = 0; c < f; ++c) g[c] = silu(g[c]) * u[c];      // H row, no rounding
  for (int j = 0; j < d; ++j) y[j] = 0.0;
  for (int c = 0; c < f; ++c) {            // c ascending for every output column j
    const double hc = g[c];
    const uint16_t* wd = Wd + static_cast<size_t>(c) * d;
    for (int j = 0; j < d; ++j) y[j] += hc * widen_bf16(wd[j]);
  }
}

}  // namespace

extern "C" {

int bgo_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// (a1) router logits.  hidden bf16 [T,d]; W_r fp32 [d,E]; b_r fp32 [E] or NULL; logits fp32 [T,E].
int bgo_router_logits(const uint16_t* hidden, const float* W_r, const float* b_r,
                      int T, int d, int E, float* logits) {
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t) {
    for (int e = 0; e < E; ++e) {
      double acc = 0.0;
      for (int j = 0; j < d; ++j)
        acc += widen_bf16(hidden[static_cast<size_t>(t) * d + j]) *
               static_cast<double>(W_r[static_cast<size_t>(j) * E + e]);
      if (b_r) acc += static_cast<double>(b_r[e]);
      logits[static_cast<size_t>(t) * E + e] = static_cast<float>(acc);
    }
  }
  return 0;
}

// (a2) top-k + softmax-renormalised gates from fp32 logits.
int bgo_topk_gate(const float* logits, int T, int E, int k, int32_t* idx, float* w) {
  if (k < 1 || k > E) return -1;
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t)
    topk_one(logits + static_cast<size_t>(t) * E, E, k, idx + static_cast<size_t>(t) * k,
             w + static_cast<size_t>(t) * k);
  return 0;
}

// (a3,a4,a5) histogram, exclusive scan, stable counting sort by expert.
int bgo_hist_scan_perm(const int32_t* idx, int T, int k, int E, int32_t* counts,
                       int32_t* offsets, int32_t* row_src, int32_t* inv_perm) {
  const int64_t R = static_cast<int64_t>(T) * k;
  for (int e = 0; e < E; ++e) counts[e] = 0;
  for (int64_t i = 0; i < R; ++i) {
    if (idx[i] < 0 || idx[i] >= E) return -1;
    counts[idx[i]] += 1;
  }
  offsets[0] = 0;
  for (int e = 0; e < E; ++e) offsets[e + 1] = offsets[e] + counts[e];
  std::vector<int32_t> cursor(offsets, offsets + E);
  for (int64_t i = 0; i < R; ++i) {        // ascending flat index => stable inside each expert
    const int32_t r = cursor[idx[i]]++;
    row_src[r] = static_cast<int32_t>(i);
    inv_perm[i] = r;
  }
  return 0;
}

// (a6) gather into expert-contiguous rows.
int bgo_gather(const uint16_t* hidden, const int32_t* row_src, int T, int k, int d, uint16_t* x_perm) {
  const int64_t R = static_cast<int64_t>(T) * k;
  for (int64_t r = 0; r < R; ++r)
    std::memcpy(x_perm + r * d, hidden + static_cast<int64_t>(row_src[r] / k) * d, sizeof(uint16_t) * d);
  return 0;
}

// (a7,a8) grouped SwiGLU expert FFN over expert-contiguous rows, unweighted, fp64 output.
int bgo_expert_ffn(const uint16_t* x_perm, const int32_t* offsets, const uint16_t* W_gate,
                   const uint16_t* W_up, const uint16_t* W_down, int R, int d, int f, int E,
                   double* y_perm) {
  if (offsets[0] != 0 || offsets[E] != R) return -1;
  for (int e = 0; e < E; ++e) {
    const uint16_t* Wg = W_gate + static_cast<size_t>(e) * d * f;
    const uint16_t* Wu = W_up + static_cast<size_t>(e) * d * f;
    const uint16_t* Wd = W_down + static_cast<size_t>(e) * f * d;
#pragma omp parallel
    {
      std::vector<double> x(d), g(f), u(f);
#pragma omp for schedule(dynamic, 1)
      for (int r = offsets[e]; r < offsets[e + 1]; ++r) {
        for (int j = 0; j < d; ++j) x[j] = widen_bf16(x_perm[static_cast<size_t>(r) * d + j]);
        expert_row(x.data(), Wg, Wu, Wd, d, f, g.data(), u.data(), y_perm + static_cast<size_t>(r) * d);
      }
    }
  }
  return 0;
}

// (a9) gate-weighted un-permute: out[t,:] = sum_s w[t,s] * y_perm[inv_perm[t*k+s],:], slot order.
int bgo_unpermute(const double* y_perm, const int32_t* inv_perm, const float* w, int T, int k,
                  int d, double* out) {
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t) {
    double* o = out + static_cast<size_t>(t) * d;
    for (int j = 0; j < d; ++j) o[j] = 0.0;
    for (int s = 0; s < k; ++s) {
      const double ws = static_cast<double>(w[static_cast<size_t>(t) * k + s]);
      const double* y = y_perm + static_cast<size_t>(inv_perm[static_cast<size_t>(t) * k + s]) * d;
      for (int j = 0; j < d; ++j) o[j] += ws * y[j];
    }
  }
  return 0;
}

// Whole layer, batched form: route -> permute -> per-expert loops -> un-permute.
// logits_in (fp32 [T,E]) may be given to skip (a1) (reading S5); routing outputs may be NULL.
int bgo_forward_batched(const uint16_t* hidden, const float* W_r, const float* b_r,
                        const uint16_t* W_gate, const uint16_t* W_up, const uint16_t* W_down,
                        int T, int d, int E, int k, int f, const float* logits_in,
                        float* logits_out, int32_t* idx_out, float* w_out, int32_t* counts_out,
                        int32_t* offsets_out, int32_t* row_src_out, int32_t* inv_perm_out,
                        double* out) {
  const size_t R = static_cast<size_t>(T) * k;
  std::vector<float> logits(static_cast<size_t>(T) * E), w(R);
  std::vector<int32_t> idx(R), counts(E), offsets(E + 1), row_src(R), inv_perm(R);
  if (logits_in) std::copy(logits_in, logits_in + logits.size(), logits.begin());
  else bgo_router_logits(hidden, W_r, b_r, T, d, E, logits.data());
  int rc = bgo_topk_gate(logits.data(), T, E, k, idx.data(), w.data());
  if (rc) return rc;
  rc = bgo_hist_scan_perm(idx.data(), T, k, E, counts.data(), offsets.data(), row_src.data(), inv_perm.data());
  if (rc) return rc;
  std::vector<uint16_t> x_perm(R * d);
  bgo_gather(hidden, row_src.data(), T, k, d, x_perm.data());
  std::vector<double> y_perm(R * d);
  rc = bgo_expert_ffn(x_perm.data(), offsets.data(), W_gate, W_up, W_down, static_cast<int>(R), d, f, E, y_perm.data());
  if (rc) return rc;
  bgo_unpermute(y_perm.data(), inv_perm.data(), w.data(), T, k, d, out);
  if (logits_out) std::copy(logits.begin(), logits.end(), logits_out);
  if (idx_out) std::copy(idx.begin(), idx.end(), idx_out);
  if (w_out) std::copy(w.begin(), w.end(), w_out);
  if (counts_out) std::copy(counts.begin(), counts.end(), counts_out);
  if (offsets_out) std::copy(offsets.begin(), offsets.end(), offsets_out);
  if (row_src_out) std::copy(row_src.begin(), row_src.end(), row_src_out);
  if (inv_perm_out) std::copy(inv_perm.begin(), inv_perm.end(), inv_perm_out);
  return 0;
}

// Whole layer, per-token brute force (the plain definition; no histogram, no permutation):
// for each listed token t: logits (or row t of logits_in), top-k, then
// out[i,:] = sum_s w_s * FFN_{e_s}(x_t).  tokens: n_tok indices into [0,T); out: fp64 [n_tok,d].
int bgo_forward_tokens(const uint16_t* hidden, const float* W_r, const float* b_r,
                       const uint16_t* W_gate, const uint16_t* W_up, const uint16_t* W_down,
                       int T, int d, int E, int k, int f, const int32_t* tokens, int n_tok,
                       const float* logits_in, double* out) {
  if (k < 1 || k > E) return -1;
  int bad = 0;
#pragma omp parallel
  {
    std::vector<double> x(d), g(f), u(f), y(d);
    std::vector<float> L(E), w(k);
    std::vector<int32_t> idx(k);
#pragma omp for schedule(dynamic, 1)
    for (int i = 0; i < n_tok; ++i) {
      const int t = tokens[i];
      if (t < 0 || t >= T) {
#pragma omp atomic write
        bad = 1;
        continue;
      }
      for (int j = 0; j < d; ++j) x[j] = widen_bf16(hidden[static_cast<size_t>(t) * d + j]);
      if (logits_in) {
        for (int e = 0; e < E; ++e) L[e] = logits_in[static_cast<size_t>(t) * E + e];
      } else {
        for (int e = 0; e < E; ++e) {
          double acc = 0.0;
          for (int j = 0; j < d; ++j) acc += x[j] * static_cast<double>(W_r[static_cast<size_t>(j) * E + e]);
          if (b_r) acc += static_cast<double>(b_r[e]);
          L[e] = static_cast<float>(acc);
        }
      }
      topk_one(L.data(), E, k, idx.data(), w.data());
      double* o = out + static_cast<size_t>(i) * d;
      for (int j = 0; j < d; ++j) o[j] = 0.0;
      for (int s = 0; s < k; ++s) {
        const int e = idx[s];
        expert_row(x.data(), W_gate + static_cast<size_t>(e) * d * f, W_up + static_cast<size_t>(e) * d * f,
                   W_down + static_cast<size_t>(e) * f * d, d, f, g.data(), u.data(), y.data());
        const double ws = static_cast<double>(w[s]);
        for (int j = 0; j < d; ++j) o[j] += ws * y[j];
      }
    }
  }
  return bad ? -1 : 0;
}

}  // extern "C"
