// oracle/haste_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded fp64 CPU statement of what the HASTE hot path
// computes (arxiv/paper_2606_01117): the group-shared fixed fan-in sparse output
// layer, its BCE-with-logits objective and its gradients, plus the dense head.
// Written from the paper's definitions only; shares no code, header, table or
// constant with the CUDA path under paper_2606_01117_b200/csrc.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library.
//
// Notation (paper symbol -> this file):  H -> d (feature dim), F -> K (fan-in per
// group), number of groups K_paper -> NG = ceil(L/G), I_k -> row g of idx[NG,K],
// w_l -> row l of W[L,K], h -> row of X[B,d].
//
// Definitions realised here (all sums in fp64, in the order written):
//   z[i,l]  = bias[l] + sum_j W[l,j] * X[i, idx[g(l), j]],  g(l) = floor(l/G)
//   y[i,l]  = 1 iff (label_offset + l) is in row i of the CSR targets
//   loss    = s * sum_i sum_l ( softplus(z[i,l]) - y[i,l]*z[i,l] )             (Eq. 3;
//             BCE(y, sigma(a)) written in its with-logits form, reading R5; s = 1/B, R1)
//   dY[i,l] = s * ( sigma(z[i,l]) - y[i,l] )                                    (derivative of the above)
//   dW[l,j] = sum_i dY[i,l] * X[i, idx[g(l), j]]
//   db[l]   = sum_i dY[i,l]
//   dX[i,f] = sum_l sum_{j : idx[g(l),j] = f} dY[i,l] * W[l,j]
//   head:   z = b_h + X_h * W_h^T ; same loss/dY ; dW_h = dY^T X_h ; dX_h = dY W_h
//
// Inputs are float32 arrays holding the values both sides consume (for bf16
// configs: the bf16-rounded values widened exactly); every product and sum is
// fp64.  No bf16 rounding of any intermediate is emulated.
//
// Two independent statements are provided:
//   O2  haste_oracle_tail_*      direct sparse definition, label-major streaming
//   O1  haste_oracle_bruteforce  scatter (idx, W) into a dense masked W_full[L,d]
//                                and run an ordinary dense layer (tiny inputs only)
// Pins (tests/test_oracle_pins.py): O1==O2, G=1 per-label loop, K=d dense layer,
// central finite differences, W=0 closed form, closed-form logits (ln 3 -> 3/4,
// ln 4), Euler identities, slot permutation, duplicate additivity.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC (oracle/build.py).

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#include <utility>

namespace {

// softplus(z) = max(z,0) + log1p(exp(-|z|))  -- the overflow-free form of log(1+e^z).
inline double softplus(double z) { return std::max(z, 0.0) + std::log1p(std::exp(-std::fabs(z))); }

// sigma(z) = 1/(1+e^-z), evaluated without overflow on either side.
inline double sigmoid(double z) {
  if (z >= 0.0) return 1.0 / (1.0 + std::exp(-z));
  const double e = std::exp(z);
  return e / (1.0 + e);
}

// Multi-hot targets of one label column: y[i] = 1 iff global id (label_offset + l)
// appears in CSR row i.  Plain scan of the row; a repeated id counts once (R7).
inline void target_column(int B, const int32_t* rowptr, const int32_t* col, int64_t gid, std::vector<double>& y) {
  for (int i = 0; i < B; ++i) {
    double v = 0.0;
    for (int32_t p = rowptr[i]; p < rowptr[i + 1]; ++p)
      if ((int64_t)col[p] == gid) v = 1.0;
    y[i] = v;
  }
}

// The (row,label) pairs of the CSR restricted to this layer, sorted by label then row.
// Used by the streaming O2 so that a pass over L labels does not rescan the CSR L times.
std::vector<std::pair<int64_t, int>> pairs_by_label(int B, const int32_t* rowptr, const int32_t* col,
                                                    int64_t label_offset, int64_t L) {
  std::vector<std::pair<int64_t, int>> pr;
  for (int i = 0; i < B; ++i)
    for (int32_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      const int64_t l = (int64_t)col[p] - label_offset;
      if (l >= 0 && l < L) pr.emplace_back(l, i);
    }
  std::sort(pr.begin(), pr.end());
  pr.erase(std::unique(pr.begin(), pr.end()), pr.end());
  return pr;
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------
// O2: sparse tail, forward + loss (+ optional logits z and dY, both [B,L] row-major fp64).
// Returns 0, or -1 if an index is outside [0,d).
// ---------------------------------------------------------------------------
int haste_oracle_tail_forward(int B, int d, int64_t L, int G, int K,
                              const float* X, const int32_t* idx, const float* W, const float* bias,
                              const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                              double* loss_out, double* z_out, double* dY_out) {
  const auto pr = pairs_by_label(B, rowptr, col, label_offset, L);
  size_t pp = 0;
  std::vector<double> y(B);
  double loss = 0.0;
  for (int64_t l = 0; l < L; ++l) {
    const int64_t g = l / G;                       // g(l)
    const int32_t* I = idx + g * (int64_t)K;       // I_g
    const float* w = W + l * (int64_t)K;           // w_l
    std::fill(y.begin(), y.end(), 0.0);
    while (pp < pr.size() && pr[pp].first == l) { y[pr[pp].second] = 1.0; ++pp; }
    for (int i = 0; i < B; ++i) {
      double z = bias ? (double)bias[l] : 0.0;
      for (int j = 0; j < K; ++j) {
        const int32_t f = I[j];
        if (f < 0 || f >= d) return -1;
        z += (double)w[j] * (double)X[(int64_t)i * d + f];     // <w_l, h_{I_g}>
      }
      loss += softplus(z) - y[i] * z;                          // Eq. 3 summand
      if (z_out) z_out[(int64_t)i * L + l] = z;
      if (dY_out) dY_out[(int64_t)i * L + l] = s * (sigmoid(z) - y[i]);
    }
  }
  if (loss_out) *loss_out = s * loss;
  return 0;
}

// O2: sparse tail backward from a given dY [B,L] fp64 (row-major).
// dW [L,K], db [L] (nullable), dX [B,d] are overwritten.
int haste_oracle_tail_backward(int B, int d, int64_t L, int G, int K,
                               const float* X, const int32_t* idx, const float* W, const double* dY,
                               double* dW, double* db, double* dX) {
  if (dX) std::fill(dX, dX + (int64_t)B * d, 0.0);
  for (int64_t l = 0; l < L; ++l) {
    const int64_t g = l / G;
    const int32_t* I = idx + g * (int64_t)K;
    const float* w = W + l * (int64_t)K;
    if (db) {
      double acc = 0.0;
      for (int i = 0; i < B; ++i) acc += dY[(int64_t)i * L + l];
      db[l] = acc;
    }
    for (int j = 0; j < K; ++j) {
      const int32_t f = I[j];
      if (f < 0 || f >= d) return -1;
      if (dW) {
        double acc = 0.0;                                             // dW_g = dZ_g^T H_g
        for (int i = 0; i < B; ++i) acc += dY[(int64_t)i * L + l] * (double)X[(int64_t)i * d + f];
        dW[l * (int64_t)K + j] = acc;
      }
      if (dX)                                                         // dh_{:,I_g} += dZ_g W_g
        for (int i = 0; i < B; ++i) dX[(int64_t)i * d + f] += dY[(int64_t)i * L + l] * (double)w[j];
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------
// O1: brute force over the dense masked matrix W_full [L,d] (tiny inputs only).
// W_full[l, idx[g(l),j]] += W[l,j]  (duplicates add, reading R4), then an ordinary
// dense layer.  Every output pointer may be NULL.  Target matrix built by a direct
// scan of each CSR row (no shared helper with O2's streaming path).
// ---------------------------------------------------------------------------
int haste_oracle_bruteforce(int B, int d, int64_t L, int G, int K,
                            const float* X, const int32_t* idx, const float* W, const float* bias,
                            const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                            double* loss_out, double* z_out, double* dY_out,
                            double* dW_out, double* db_out, double* dX_out) {
  std::vector<double> Wf((size_t)L * d, 0.0);
  for (int64_t l = 0; l < L; ++l)
    for (int j = 0; j < K; ++j) {
      const int32_t f = idx[(l / G) * (int64_t)K + j];
      if (f < 0 || f >= d) return -1;
      Wf[(size_t)l * d + f] += (double)W[l * (int64_t)K + j];
    }
  std::vector<double> Y((size_t)B * L, 0.0);
  for (int i = 0; i < B; ++i)
    for (int32_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      const int64_t l = (int64_t)col[p] - label_offset;
      if (l >= 0 && l < L) Y[(size_t)i * L + l] = 1.0;
    }
  std::vector<double> Z((size_t)B * L), dY((size_t)B * L);
  double loss = 0.0;
  for (int i = 0; i < B; ++i)
    for (int64_t l = 0; l < L; ++l) {
      double z = bias ? (double)bias[l] : 0.0;
      for (int f = 0; f < d; ++f) z += (double)X[(size_t)i * d + f] * Wf[(size_t)l * d + f];
      Z[(size_t)i * L + l] = z;
      loss += softplus(z) - Y[(size_t)i * L + l] * z;
      dY[(size_t)i * L + l] = s * (sigmoid(z) - Y[(size_t)i * L + l]);
    }
  if (loss_out) *loss_out = s * loss;
  if (z_out) std::copy(Z.begin(), Z.end(), z_out);
  if (dY_out) std::copy(dY.begin(), dY.end(), dY_out);
  if (dX_out)
    for (int i = 0; i < B; ++i)
      for (int f = 0; f < d; ++f) {
        double acc = 0.0;
        for (int64_t l = 0; l < L; ++l) acc += dY[(size_t)i * L + l] * Wf[(size_t)l * d + f];
        dX_out[(size_t)i * d + f] = acc;
      }
  if (dW_out || db_out) {
    std::vector<double> dWf((size_t)L * d, 0.0);
    for (int64_t l = 0; l < L; ++l)
      for (int f = 0; f < d; ++f) {
        double acc = 0.0;
        for (int i = 0; i < B; ++i) acc += dY[(size_t)i * L + l] * (double)X[(size_t)i * d + f];
        dWf[(size_t)l * d + f] = acc;
      }
    if (dW_out)
      for (int64_t l = 0; l < L; ++l)
        for (int j = 0; j < K; ++j)
          dW_out[l * (int64_t)K + j] = dWf[(size_t)l * d + idx[(l / G) * (int64_t)K + j]];
    if (db_out)
      for (int64_t l = 0; l < L; ++l) {
        double acc = 0.0;
        for (int i = 0; i < B; ++i) acc += dY[(size_t)i * L + l];
        db_out[l] = acc;
      }
  }
  return 0;
}

// ---------------------------------------------------------------------------
// Dense head: z = b + X W_h^T, same objective; dW_h = dY^T X; dX = dY W_h.
// ---------------------------------------------------------------------------
int haste_oracle_head_forward(int B, int d, int64_t Lh, const float* X, const float* Wh, const float* bias,
                              const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                              double* loss_out, double* z_out, double* dY_out) {
  std::vector<double> y(B);
  double loss = 0.0;
  for (int64_t l = 0; l < Lh; ++l) {
    target_column(B, rowptr, col, label_offset + l, y);
    for (int i = 0; i < B; ++i) {
      double z = bias ? (double)bias[l] : 0.0;
      for (int f = 0; f < d; ++f) z += (double)Wh[l * (int64_t)d + f] * (double)X[(int64_t)i * d + f];
      loss += softplus(z) - y[i] * z;
      if (z_out) z_out[(int64_t)i * Lh + l] = z;
      if (dY_out) dY_out[(int64_t)i * Lh + l] = s * (sigmoid(z) - y[i]);
    }
  }
  if (loss_out) *loss_out = s * loss;
  return 0;
}

int haste_oracle_head_backward(int B, int d, int64_t Lh, const float* X, const float* Wh, const double* dY,
                               double* dWh, double* db, double* dX) {
  if (dWh)
    for (int64_t l = 0; l < Lh; ++l)
      for (int f = 0; f < d; ++f) {
        double acc = 0.0;
        for (int i = 0; i < B; ++i) acc += dY[(int64_t)i * Lh + l] * (double)X[(int64_t)i * d + f];
        dWh[l * (int64_t)d + f] = acc;
      }
  if (db)
    for (int64_t l = 0; l < Lh; ++l) {
      double acc = 0.0;
      for (int i = 0; i < B; ++i) acc += dY[(int64_t)i * Lh + l];
      db[l] = acc;
    }
  if (dX)
    for (int i = 0; i < B; ++i)
      for (int f = 0; f < d; ++f) {
        double acc = 0.0;
        for (int64_t l = 0; l < Lh; ++l) acc += dY[(int64_t)i * Lh + l] * (double)Wh[l * (int64_t)d + f];
        dX[(int64_t)i * d + f] = acc;
      }
  return 0;
}

// ---------------------------------------------------------------------------
// Sampled statements for full-size configs (the same definitions, evaluated one
// output at a time so a test can check a sample of a 670K- or 3M-label run).
// ---------------------------------------------------------------------------

// Logit and dY for n (row,label) pairs: z_out[n], dY_out[n] (either nullable).
int haste_oracle_tail_points(int B, int d, int64_t L, int G, int K,
                             const float* X, const int32_t* idx, const float* W, const float* bias,
                             const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                             int64_t n, const int32_t* rows, const int64_t* labels, double* z_out, double* dY_out) {
  for (int64_t t = 0; t < n; ++t) {
    const int i = rows[t];
    const int64_t l = labels[t];
    if (i < 0 || i >= B || l < 0 || l >= L) return -1;
    const int32_t* I = idx + (l / G) * (int64_t)K;
    double z = bias ? (double)bias[l] : 0.0;
    for (int j = 0; j < K; ++j) z += (double)W[l * (int64_t)K + j] * (double)X[(int64_t)i * d + I[j]];
    double y = 0.0;
    for (int32_t p = rowptr[i]; p < rowptr[i + 1]; ++p)
      if ((int64_t)col[p] == label_offset + l) y = 1.0;
    if (z_out) z_out[t] = z;
    if (dY_out) dY_out[t] = s * (sigmoid(z) - y);
  }
  return 0;
}

// For n sampled labels: the label's dY column [n,B], its dW row [n,K] and db [n]
// (fp64 end to end: dY is the exact one, not a rounded copy).
int haste_oracle_tail_label_rows(int B, int d, int64_t L, int G, int K,
                                 const float* X, const int32_t* idx, const float* W, const float* bias,
                                 const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                                 int64_t n, const int64_t* labels, double* dYcol_out, double* dW_out, double* db_out) {
  std::vector<double> y(B), dy(B);
  for (int64_t t = 0; t < n; ++t) {
    const int64_t l = labels[t];
    if (l < 0 || l >= L) return -1;
    const int32_t* I = idx + (l / G) * (int64_t)K;
    target_column(B, rowptr, col, label_offset + l, y);
    for (int i = 0; i < B; ++i) {
      double z = bias ? (double)bias[l] : 0.0;
      for (int j = 0; j < K; ++j) z += (double)W[l * (int64_t)K + j] * (double)X[(int64_t)i * d + I[j]];
      dy[i] = s * (sigmoid(z) - y[i]);
      if (dYcol_out) dYcol_out[t * B + i] = dy[i];
    }
    if (dW_out)
      for (int j = 0; j < K; ++j) {
        double acc = 0.0;
        for (int i = 0; i < B; ++i) acc += dy[i] * (double)X[(int64_t)i * d + I[j]];
        dW_out[t * K + j] = acc;
      }
    if (db_out) {
      double acc = 0.0;
      for (int i = 0; i < B; ++i) acc += dy[i];
      db_out[t] = acc;
    }
  }
  return 0;
}

// For n sampled batch rows: the row's loss contribution (unscaled by nothing: it is
// s * sum_l (softplus - y z)), and its full dX row [n,d], summing over ALL labels.
int haste_oracle_tail_batch_rows(int B, int d, int64_t L, int G, int K,
                                 const float* X, const int32_t* idx, const float* W, const float* bias,
                                 const int32_t* rowptr, const int32_t* col, int64_t label_offset, double s,
                                 int64_t n, const int32_t* rows, double* loss_rows_out, double* dX_out) {
  for (int64_t t = 0; t < n; ++t) {
    const int i = rows[t];
    if (i < 0 || i >= B) return -1;
    std::vector<char> pos((size_t)L, 0);
    for (int32_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      const int64_t l = (int64_t)col[p] - label_offset;
      if (l >= 0 && l < L) pos[(size_t)l] = 1;
    }
    double loss = 0.0;
    if (dX_out) std::fill(dX_out + t * d, dX_out + (t + 1) * d, 0.0);
    for (int64_t l = 0; l < L; ++l) {
      const int32_t* I = idx + (l / G) * (int64_t)K;
      double z = bias ? (double)bias[l] : 0.0;
      for (int j = 0; j < K; ++j) z += (double)W[l * (int64_t)K + j] * (double)X[(int64_t)i * d + I[j]];
      const double y = pos[(size_t)l] ? 1.0 : 0.0;
      loss += softplus(z) - y * z;
      const double dy = s * (sigmoid(z) - y);
      if (dX_out)
        for (int j = 0; j < K; ++j) dX_out[t * d + I[j]] += dy * (double)W[l * (int64_t)K + j];
    }
    if (loss_rows_out) loss_rows_out[t] = s * loss;
  }
  return 0;
}

// ---------------------------------------------------------------------------
// Optimizer step of the output layer: "SGD with momentum for the final layer".
// The paper names the method and nothing else (no dampening, Nesterov or weight-decay statement), so this is the
// textbook heavy-ball form, reading R13:
//     g' = g + wd * w          (L2 weight decay, wd = 0 turns it off)
//     v  <- mu * v + g'        (momentum buffer, starts at 0)
//     w  <- w - lr * v
// applied element by element to n parameters, everything in fp64.  Pins (tests/test_oracle_pins.py): mu = 0 is plain
// gradient descent; two and n steps on a constant gradient have closed forms (w_n = w_0 - lr g sum_{t<n} (1-mu^{t+1})/(1-mu));
// g = 0, mu = 0 shrinks w by (1 - lr wd).
// ---------------------------------------------------------------------------
int haste_oracle_sgd_momentum(int64_t n, const double* w, const double* g, const double* v, double lr, double mu, double wd,
                              double* w_out, double* v_out) {
  for (int64_t e = 0; e < n; ++e) {
    const double gp = g[e] + wd * w[e];
    const double vn = mu * v[e] + gp;
    v_out[e] = vn;
    w_out[e] = w[e] - lr * vn;
  }
  return 0;
}

// ---------------------------------------------------------------------------
// Group-shared rewiring, Algorithm 3, SURVEY.md 8(f3).  Step by step in the paper's order:
//   1. scores   S[k,j] = mean over the labels l of group k of |w_l[j]|
//   2. m = floor(NG * K * rho); mask M = the m smallest entries of S
//   3. regrow   I_k[j] <- Unif{0..H-1} for every masked (k,j)
//   4. reinit   w_l[j] <- 0  (zero mode)  or  Unif(-1/sqrt(F), 1/sqrt(F))  (random mode)
// Readings (R15): a score decides an INTEGER (which slots are pruned), so it is computed the way the kernel
// computes it -- fp32, labels added in ascending order, divided by the label count -- and ties are broken by the flat
// index k*K + j (smaller first); the partial last group averages over the labels it has.  Random numbers come from a
// counter-based generator both sides implement (SplitMix64 finaliser of seed + golden-ratio * (counter + 1)):
//   regrown feature  u = floor(d * h / 2^64) = high 64 bits of h * d,      h = mix(seed, k*K + j)
//   random weight    w = float(2 U - 1) * float(1/sqrt(K)) in fp32, U = (h >> 41) / 2^23,  h = mix(seed ^ 0x5851f42d4c957f2d, l*K + j)
//                    (then rounded to bf16 by the caller when the layer stores bf16)
// Optional extras, not in the paper (its Alg. 3 stops after step 4): momentum entries of reinitialised weights are set
// to 0; `resort` != 0 re-sorts every touched idx row ascending (stable: ties keep their slot order) and permutes the W
// (and momentum) columns of the group's labels with it -- the layer's function is invariant under slot permutations
// (pin P8), and sorted rows are what the tcgen05 dX kernel's on-chip classes need.
// ---------------------------------------------------------------------------
static inline uint64_t rw_mix(uint64_t seed, uint64_t counter) {
  uint64_t z = seed + 0x9e3779b97f4a7c15ULL * (counter + 1);
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ULL;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebULL;
  return z ^ (z >> 31);
}
uint64_t haste_oracle_rewire_mix(uint64_t seed, uint64_t counter) { return rw_mix(seed, counter); }

// scores_out [NG*K] fp32 (optional), mask_out [NG*K] bytes (optional).  W, mom are float32 arrays updated in place
// (W holds the layer's values widened; the caller re-rounds random weights to the storage type).  Returns m, or -1.
int64_t haste_oracle_rewire(int64_t L, int G, int K, int d, int32_t* idx, float* W, float* mom, double rho, int init_random,
                            uint64_t seed, int resort, float* scores_out, unsigned char* mask_out) {
  const int64_t NG = (L + G - 1) / G, n = NG * K;
  std::vector<float> S((size_t)n);
  for (int64_t k = 0; k < NG; ++k) {
    const int64_t l0 = k * G, l1 = std::min<int64_t>(L, l0 + G);
    for (int j = 0; j < K; ++j) {
      float acc = 0.f;
      for (int64_t l = l0; l < l1; ++l) acc = acc + std::fabs(W[l * K + j]);
      S[(size_t)(k * K + j)] = acc / (float)(l1 - l0);
    }
  }
  if (scores_out) std::copy(S.begin(), S.end(), scores_out);
  const int64_t m = (int64_t)std::floor((double)n * rho);
  std::vector<unsigned char> M((size_t)n, 0);
  if (m > 0) {
    std::vector<int64_t> order((size_t)n);
    for (int64_t e = 0; e < n; ++e) order[(size_t)e] = e;
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return S[(size_t)a] < S[(size_t)b]; });
    for (int64_t t = 0; t < m && t < n; ++t) M[(size_t)order[(size_t)t]] = 1;
  }
  if (mask_out) std::copy(M.begin(), M.end(), mask_out);
  if (m <= 0) return 0;
  const float r32 = (float)(1.0 / std::sqrt((double)K));
  for (int64_t k = 0; k < NG; ++k) {
    bool touched = false;
    for (int j = 0; j < K; ++j) {
      if (!M[(size_t)(k * K + j)]) continue;
      touched = true;
      const uint64_t h = rw_mix(seed, (uint64_t)(k * K + j));
      idx[k * K + j] = (int32_t)(uint64_t)(((unsigned __int128)h * (unsigned __int128)(uint64_t)d) >> 64);
      const int64_t l0 = k * G, l1 = std::min<int64_t>(L, l0 + G);
      for (int64_t l = l0; l < l1; ++l) {
        float w = 0.f;
        if (init_random) {
          const uint64_t hw = rw_mix(seed ^ 0x5851f42d4c957f2dULL, (uint64_t)(l * K + j));
          const float a = (float)(2.0 * ((double)(hw >> 41) * (1.0 / 8388608.0)) - 1.0);
          w = a * r32;
        }
        W[l * K + j] = w;
        if (mom) mom[l * K + j] = 0.f;
      }
    }
    if (touched && resort) {
      std::vector<int> perm((size_t)K);
      for (int j = 0; j < K; ++j) perm[(size_t)j] = j;
      std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return idx[k * K + a] < idx[k * K + b]; });
      std::vector<int32_t> irow((size_t)K);
      for (int j = 0; j < K; ++j) irow[(size_t)j] = idx[k * K + perm[(size_t)j]];
      for (int j = 0; j < K; ++j) idx[k * K + j] = irow[(size_t)j];
      const int64_t l0 = k * G, l1 = std::min<int64_t>(L, l0 + G);
      std::vector<float> row((size_t)K);
      for (int64_t l = l0; l < l1; ++l) {
        for (int j = 0; j < K; ++j) row[(size_t)j] = W[l * K + perm[(size_t)j]];
        for (int j = 0; j < K; ++j) W[l * K + j] = row[(size_t)j];
        if (mom) {
          for (int j = 0; j < K; ++j) row[(size_t)j] = mom[l * K + perm[(size_t)j]];
          for (int j = 0; j < K; ++j) mom[l * K + j] = row[(size_t)j];
        }
      }
    }
  }
  return m;
}

// Scalar helpers exported so pins can check them against closed forms directly.
double haste_oracle_softplus(double z) { return softplus(z); }
double haste_oracle_sigmoid(double z) { return sigmoid(z); }

}  // extern "C"
