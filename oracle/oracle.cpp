// oracle/oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library.  It shares no code, header, table or helper with the CUDA path
// (paper_2606_11169_b200/csrc) and neither includes the other.
//
// What it is: the plain definition of the single-device expert-parallel MoE chunk named by
// BASELINE.json:north_star, written out as slow, obviously-correct loops with fp64 arithmetic.
// PAPER.md is silent on the MoE math (its only MoE text is Listing 1, PAPER.md:157-165:
// `self.router(x)`, `self.experts(x)`), so every formula below follows SURVEY.md §8(c)
// "Definition" items 1-5, which restate BASELINE.json:north_star / configs; the one part where
// PAPER.md is the authority, the list scheduler of §4.3.1 and the
// event rule of §4.3.2, is restated in oracle_list_schedule().
//
// Conventions: row-major contiguous host arrays.  Inputs that the GPU also consumes (x, dY,
// weights) come as `const void*` + dtype (0 = fp32, 1 = bf16 bit patterns) and are widened
// exactly to fp64; logits are fp32.  Every floating-point result is fp64 and is never rounded.
// Integer results are int32.  Return value 0 = ok, negative = precondition violated.
//
// Pins (tests/test_oracle_*.py): invariants, closed forms, torch CPU fp64 special cases, dense
// brute force, finite differences, hand-derived scheduler golden order (tests/golden/).
// Nothing here is "parity unpinned" except the choice among readings c-2..c-5, c-14, c-20
// (SURVEY.md §8c), which only BASELINE.json's own claims pin; see DESIGN.md.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

struct Desc {  // mirrors oracle.py: OracleDesc
    int32_t T, d, E, k, e_lo, E_loc, I, dtype, gate_mode, row_align;
};

inline double ld(const void* p, int dtype, size_t i) {
    if (dtype == 0) return (double)static_cast<const float*>(p)[i];
    uint32_t u = (uint32_t)static_cast<const uint16_t*>(p)[i] << 16;  // bf16 -> fp32, exact
    float f;
    std::memcpy(&f, &u, 4);
    return (double)f;
}

inline double sigmoid(double v) { return 1.0 / (1.0 + std::exp(-v)); }

int g_threads = 1;

}  // namespace

extern "C" {

// Threads used by the row loops of the FFN functions (independent rows).
void oracle_set_threads(int n) { g_threads = n < 1 ? 1 : n; }
int oracle_get_threads() { return g_threads; }

// ---------------------------------------------------------------------------------------------
// 0. Router (Listing 1 `self.router(x)`; readings c-5, c-18): the step before F1.
//    z[t,e] = sum_i x[t,i] W_r[i,e] + bias[e], in fp64 and unrounded (the generator's logits are this sum rounded to
//    fp32 followed by one fp32 add of the bias).  Backward (Definition 5, last sentence): dW_r[i,e] = sum_t x[t,i]
//    dz[t,e] and the router's part of dX, dX_r[t,i] = sum_e dz[t,e] W_r[i,e], for a dense dz [T,E].
int oracle_router_fwd(const Desc* D, const void* x, const void* w_r, const float* bias, double* z) {
    const int T = D->T, d = D->d, E = D->E;
    for (int t = 0; t < T; ++t)
        for (int e = 0; e < E; ++e) {
            double acc = 0.0;
            for (int i = 0; i < d; ++i) acc += ld(x, D->dtype, (size_t)t * d + i) * ld(w_r, D->dtype, (size_t)i * E + e);
            z[(size_t)t * E + e] = acc + (bias ? (double)bias[e] : 0.0);
        }
    return 0;
}
int oracle_router_bwd(const Desc* D, const void* x, const void* w_r, const double* dz, double* dw_r, double* dx_r) {
    const int T = D->T, d = D->d, E = D->E;
    for (int i = 0; i < d; ++i)
        for (int e = 0; e < E; ++e) {
            double acc = 0.0;
            for (int t = 0; t < T; ++t) acc += ld(x, D->dtype, (size_t)t * d + i) * dz[(size_t)t * E + e];
            dw_r[(size_t)i * E + e] = acc;
        }
    for (int t = 0; t < T; ++t)
        for (int i = 0; i < d; ++i) {
            double acc = 0.0;
            for (int e = 0; e < E; ++e) acc += dz[(size_t)t * E + e] * ld(w_r, D->dtype, (size_t)i * E + e);
            dx_r[(size_t)t * d + i] = acc;
        }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// 1. Routing (SURVEY.md §8c Definition 1; BASELINE.json:north_star part 1; tie rule c-6; c-7).
//    topk_idx[t, 0..k) = the k experts with the largest logits, ties to the lowest index,
//    listed by descending logit.  gates: mode 0 softmax over the selected k, mode 1 sigmoid
//    normalised over the selected k, mode 2 softmax over all E (not renormalised).
//    counts_global[e] = number of (t, j) with topk_idx[t, j] = e.
// ---------------------------------------------------------------------------------------------
int oracle_route_topk(const Desc* D, const float* z, int32_t* topk_idx, double* gates, int32_t* counts_global) {
    const int T = D->T, E = D->E, k = D->k;
    if (E < 1 || k < 1 || k > E) return -1;
    for (int e = 0; e < E; ++e) counts_global[e] = 0;
    std::vector<char> used((size_t)E, 0);
    for (int t = 0; t < T; ++t) {
        const float* zt = z + (size_t)t * E;
        int finite = 0;
        for (int e = 0; e < E; ++e) {
            if (std::isnan(zt[e]) || zt[e] == INFINITY) return -2;  // c-7: finite or -inf only
            if (std::isfinite(zt[e])) ++finite;
        }
        if (finite < k) return -3;
        std::fill(used.begin(), used.end(), 0);
        for (int j = 0; j < k; ++j) {
            int best = -1;
            for (int e = 0; e < E; ++e)
                if (!used[e] && (best < 0 || zt[e] > zt[best])) best = e;  // strict > : lowest index wins ties
            used[best] = 1;
            topk_idx[(size_t)t * k + j] = best;
            counts_global[best] += 1;
        }
        const int32_t* sel = topk_idx + (size_t)t * k;
        double* g = gates + (size_t)t * k;
        if (D->gate_mode == 0) {
            double z0 = zt[sel[0]], s = 0;
            for (int j = 0; j < k; ++j) s += std::exp((double)zt[sel[j]] - z0);
            for (int j = 0; j < k; ++j) g[j] = std::exp((double)zt[sel[j]] - z0) / s;
        } else if (D->gate_mode == 1) {
            double s = 0;
            for (int j = 0; j < k; ++j) s += sigmoid(zt[sel[j]]);
            for (int j = 0; j < k; ++j) g[j] = sigmoid(zt[sel[j]]) / s;
        } else if (D->gate_mode == 2) {
            double m = zt[sel[0]], s = 0;
            for (int e = 0; e < E; ++e) s += std::exp((double)zt[e] - m);
            for (int j = 0; j < k; ++j) g[j] = std::exp((double)zt[sel[j]] - m) / s;
        } else {
            return -4;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// 2. Permutation (Definition 2; north_star part 2; readings c-8, c-9).
//    counts[i] for local expert e_lo+i; offsets[0]=0, offsets[i+1]=offsets[i]+roundup(counts[i],
//    row_align); row_of[a] = offsets[i] + #{t' < t : e in topk_idx[t']} for a=(t,j) with local
//    expert e, else -1; src_of[row_of[a]] = a, every other row (pad, tail up to a_cap) = -1.
// ---------------------------------------------------------------------------------------------
int oracle_permute(const Desc* D, const int32_t* topk_idx, int32_t a_cap, int32_t* counts, int32_t* offsets,
                   int32_t* row_of, int32_t* src_of) {
    const int T = D->T, k = D->k, EL = D->E_loc, lo = D->e_lo, al = D->row_align;
    if (al < 1) return -1;
    for (int i = 0; i < EL; ++i) counts[i] = 0;
    for (size_t a = 0; a < (size_t)T * k; ++a) {
        int i = topk_idx[a] - lo;
        if (i >= 0 && i < EL) counts[i] += 1;
    }
    offsets[0] = 0;
    for (int i = 0; i < EL; ++i) offsets[i + 1] = offsets[i] + (counts[i] + al - 1) / al * al;
    if (offsets[EL] > a_cap) return -2;
    for (int r = 0; r < a_cap; ++r) src_of[r] = -1;
    // Tokens ascending; the experts of one token are distinct, so the number of earlier tokens
    // routed to e equals the number of earlier assignments to e: a running cursor per expert.
    std::vector<int32_t> seen(EL, 0);
    for (int t = 0; t < T; ++t)
        for (int j = 0; j < k; ++j) {
            size_t a = (size_t)t * k + j;
            int i = topk_idx[a] - lo;
            if (i < 0 || i >= EL) { row_of[a] = -1; continue; }
            int r = offsets[i] + seen[i];
            seen[i] += 1;
            row_of[a] = r;
            src_of[r] = (int32_t)a;
        }
    return 0;
}

// Xp[row_of[a]] = x[t], gate_rows[row_of[a]] = gates[a]; pad rows 0 (Definition 2).
int oracle_pack(const Desc* D, const void* x, const int32_t* src_of, const double* gates, int32_t a_cap,
                double* Xp, double* gate_rows) {
    const int d = D->d, k = D->k;
    for (int r = 0; r < a_cap; ++r) {
        int a = src_of[r];
        gate_rows[r] = a < 0 ? 0.0 : gates[a];
        for (int c = 0; c < d; ++c) Xp[(size_t)r * d + c] = a < 0 ? 0.0 : ld(x, D->dtype, (size_t)(a / k) * d + c);
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// 3. Expert FFN forward on a list of rows (Definition 3; north_star part 3).
//    Row r uses expert ex[r] (index into the weight arrays; ex[r] < 0: pad row, outputs 0):
//      g = X[r] W_gate[e], u = X[r] W_up[e], h = (g / (1 + e^-g)) * u, O[r] = h W_down[e].
//    W_gate, W_up: [n_e][d][I]; W_down: [n_e][I][d].  G,U,H: [n,I]; O: [n,d]; any may be null.
// ---------------------------------------------------------------------------------------------
int oracle_ffn_fwd_rows(const Desc* D, int32_t I, int32_t n, const double* X, const int32_t* ex, const void* Wg,
                        const void* Wu, const void* Wd, double* G, double* U, double* H, double* O) {
    const int d = D->d, dt = D->dtype;
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads) if (g_threads > 1)
    for (int r = 0; r < n; ++r) {
        std::vector<double> g(I, 0.0), u(I, 0.0), h(I, 0.0), o(d, 0.0);
        const int e = ex[r];
        if (e >= 0) {
            const size_t wb = (size_t)e * d * I;
            for (int i = 0; i < d; ++i) {
                const double xi = X[(size_t)r * d + i];
                for (int j = 0; j < I; ++j) {
                    g[j] += xi * ld(Wg, dt, wb + (size_t)i * I + j);
                    u[j] += xi * ld(Wu, dt, wb + (size_t)i * I + j);
                }
            }
            for (int j = 0; j < I; ++j) h[j] = g[j] / (1.0 + std::exp(-g[j])) * u[j];
            for (int j = 0; j < I; ++j)
                for (int c = 0; c < d; ++c) o[c] += h[j] * ld(Wd, dt, wb + (size_t)j * d + c);
        }
        if (G) std::copy(g.begin(), g.end(), G + (size_t)r * I);
        if (U) std::copy(u.begin(), u.end(), U + (size_t)r * I);
        if (H) std::copy(h.begin(), h.end(), H + (size_t)r * I);
        if (O) std::copy(o.begin(), o.end(), O + (size_t)r * d);
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// 4. Combine (Definition 4; north_star part 4; readings c-10..c-12).
//    Y[t] = sum_{j: row_of[t,j] >= 0} gates[t,j] * O[row_of[t,j]]  (+ S[t] if S != null).
// ---------------------------------------------------------------------------------------------
int oracle_combine(const Desc* D, const double* O, const int32_t* row_of, const double* gates, const double* S,
                   double* Y) {
    const int T = D->T, d = D->d, k = D->k;
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < d; ++c) {
            double y = 0;
            for (int j = 0; j < k; ++j) {
                int r = row_of[(size_t)t * k + j];
                if (r >= 0) y += gates[(size_t)t * k + j] * O[(size_t)r * d + c];
            }
            if (S) y += S[(size_t)t * d + c];
            Y[(size_t)t * d + c] = y;
        }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// 5. Backward (Definition 5; north_star part 5 "combine-grad, dgrad, wgrad, unpack").
// ---------------------------------------------------------------------------------------------
// dgates[t,j] = <dY[t], O[row]> (0 if not local); dO[r] = gate_rows[r] * dY[token(r)], pad rows 0.
int oracle_combine_bwd(const Desc* D, const void* dY, const double* O, const int32_t* row_of, const int32_t* src_of,
                       const double* gate_rows, int32_t a_cap, double* dO, double* dgates) {
    const int T = D->T, d = D->d, k = D->k, dt = D->dtype;
    for (size_t a = 0; a < (size_t)T * k; ++a) {
        int r = row_of[a];
        double s = 0;
        if (r >= 0)
            for (int c = 0; c < d; ++c) s += ld(dY, dt, (a / k) * d + c) * O[(size_t)r * d + c];
        dgates[a] = s;
    }
    for (int r = 0; r < a_cap; ++r) {
        int a = src_of[r];
        for (int c = 0; c < d; ++c)
            dO[(size_t)r * d + c] = a < 0 ? 0.0 : gate_rows[r] * ld(dY, dt, (size_t)(a / k) * d + c);
    }
    return 0;
}

// Per row r with expert e = ex[r] (recomputing g, u exactly from X[r]):
//   dh = dO[r] W_down[e]^T;  s = sigma(g);  dg = dh * u * s (1 + g (1 - s));  du = dh * silu(g);
//   dX[r] = dg W_gate[e]^T + du W_up[e]^T.      Outputs dX [n,d]; dG, dU, H [n,I] (nullable).
int oracle_ffn_bwd_rows(const Desc* D, int32_t I, int32_t n, const double* X, const int32_t* ex, const double* dO,
                        const void* Wg, const void* Wu, const void* Wd, double* dX, double* dG, double* dU,
                        double* H) {
    const int d = D->d, dt = D->dtype;
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads) if (g_threads > 1)
    for (int r = 0; r < n; ++r) {
        std::vector<double> g(I, 0.0), u(I, 0.0), h(I, 0.0), dh(I, 0.0), dg(I, 0.0), du(I, 0.0), dx(d, 0.0);
        const int e = ex[r];
        if (e >= 0) {
            const size_t wb = (size_t)e * d * I;
            for (int i = 0; i < d; ++i) {
                const double xi = X[(size_t)r * d + i];
                for (int j = 0; j < I; ++j) {
                    g[j] += xi * ld(Wg, dt, wb + (size_t)i * I + j);
                    u[j] += xi * ld(Wu, dt, wb + (size_t)i * I + j);
                }
            }
            for (int j = 0; j < I; ++j) {
                double acc = 0;
                for (int c = 0; c < d; ++c) acc += dO[(size_t)r * d + c] * ld(Wd, dt, wb + (size_t)j * d + c);
                dh[j] = acc;
            }
            for (int j = 0; j < I; ++j) {
                const double s = sigmoid(g[j]);
                const double silu = g[j] * s;
                h[j] = silu * u[j];
                dg[j] = dh[j] * u[j] * s * (1.0 + g[j] * (1.0 - s));
                du[j] = dh[j] * silu;
            }
            for (int i = 0; i < d; ++i) {
                double acc = 0;
                for (int j = 0; j < I; ++j)
                    acc += dg[j] * ld(Wg, dt, wb + (size_t)i * I + j) + du[j] * ld(Wu, dt, wb + (size_t)i * I + j);
                dx[i] = acc;
            }
        }
        if (dX) std::copy(dx.begin(), dx.end(), dX + (size_t)r * d);
        if (dG) std::copy(dg.begin(), dg.end(), dG + (size_t)r * I);
        if (dU) std::copy(du.begin(), du.end(), dU + (size_t)r * I);
        if (H) std::copy(h.begin(), h.end(), H + (size_t)r * I);
    }
    return 0;
}

// dW_gate[e] = sum_r X[r]^T dG[r], dW_up[e] = sum_r X[r]^T dU[r], dW_down[e] = sum_r H[r]^T dO[r]
// over the rows with ex[r] = e; experts with no rows get exact zeros.  dW*: fp64, weight layout.
int oracle_wgrad(const Desc* D, int32_t I, int32_t n_e, int32_t n, const double* X, const int32_t* ex,
                 const double* dG, const double* dU, const double* H, const double* dO, double* dWg, double* dWu,
                 double* dWd) {
    const int d = D->d;
    const size_t per = (size_t)d * I;
    std::fill(dWg, dWg + per * n_e, 0.0);
    std::fill(dWu, dWu + per * n_e, 0.0);
    std::fill(dWd, dWd + per * n_e, 0.0);
    for (int r = 0; r < n; ++r) {
        const int e = ex[r];
        if (e < 0) continue;
        if (e >= n_e) return -1;
        for (int i = 0; i < d; ++i)
            for (int j = 0; j < I; ++j) {
                dWg[e * per + (size_t)i * I + j] += X[(size_t)r * d + i] * dG[(size_t)r * I + j];
                dWu[e * per + (size_t)i * I + j] += X[(size_t)r * d + i] * dU[(size_t)r * I + j];
            }
        for (int j = 0; j < I; ++j)
            for (int c = 0; c < d; ++c) dWd[e * per + (size_t)j * d + c] += H[(size_t)r * I + j] * dO[(size_t)r * d + c];
    }
    return 0;
}

// Column-sampled form of the same definitions for full-size configs: for the listed intermediate
// columns J (all rows use expert e): g, u, h, dh, dg, du restricted to J.  Outputs [n, nJ].
int oracle_ffn_cols(const Desc* D, int32_t I, int32_t e, int32_t n, const double* X, const double* dO, int32_t nJ,
                    const int32_t* J, const void* Wg, const void* Wu, const void* Wd, double* Hc, double* dGc,
                    double* dUc) {
    const int d = D->d, dt = D->dtype;
    const size_t wb = (size_t)e * d * I;
#pragma omp parallel for schedule(static) num_threads(g_threads) if (g_threads > 1)
    for (int r = 0; r < n; ++r)
        for (int q = 0; q < nJ; ++q) {
            const int j = J[q];
            double g = 0, u = 0, dh = 0;
            for (int i = 0; i < d; ++i) {
                g += X[(size_t)r * d + i] * ld(Wg, dt, wb + (size_t)i * I + j);
                u += X[(size_t)r * d + i] * ld(Wu, dt, wb + (size_t)i * I + j);
            }
            for (int c = 0; c < d; ++c) dh += dO[(size_t)r * d + c] * ld(Wd, dt, wb + (size_t)j * d + c);
            const double s = sigmoid(g);
            Hc[(size_t)r * nJ + q] = g * s * u;
            dGc[(size_t)r * nJ + q] = dh * u * s * (1.0 + g * (1.0 - s));
            dUc[(size_t)r * nJ + q] = dh * g * s;
        }
    return 0;
}

// dX[t] = sum_{j local} dXp[row_of[t,j]]  (+ dXs[t] if dXs != null).
int oracle_unpack(const Desc* D, const double* dXp, const int32_t* row_of, const double* dXs, double* dX) {
    const int T = D->T, d = D->d, k = D->k;
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < d; ++c) {
            double v = 0;
            for (int j = 0; j < k; ++j) {
                int r = row_of[(size_t)t * k + j];
                if (r >= 0) v += dXp[(size_t)r * d + c];
            }
            if (dXs) v += dXs[(size_t)t * d + c];
            dX[(size_t)t * d + c] = v;
        }
    return 0;
}

// Gate-normalisation backward (Definition 5, last sentence).
//   mode 0: dz_j = g_j (dgates_j - sum_j' g_j' dgates_j')                       -> dz [T,k]
//   mode 1: ds_j = (dgates_j - sum_j' g_j' dgates_j') / sum_j' s_j';  dz_j = ds_j s_j (1 - s_j)  -> dz [T,k]
//   mode 2: p = softmax(z) over all E; dz_e = sum_j dgates_j p_{e_j} ([e = e_j] - p_e)           -> dz [T,E]
int oracle_route_bwd(const Desc* D, const float* z, const int32_t* topk_idx, const double* dgates, double* dz) {
    const int T = D->T, E = D->E, k = D->k;
    for (int t = 0; t < T; ++t) {
        const float* zt = z + (size_t)t * E;
        const int32_t* sel = topk_idx + (size_t)t * k;
        const double* dgt = dgates + (size_t)t * k;
        if (D->gate_mode == 0) {
            std::vector<double> g(k);
            double z0 = zt[sel[0]], s = 0, dot = 0;
            for (int j = 0; j < k; ++j) s += std::exp((double)zt[sel[j]] - z0);
            for (int j = 0; j < k; ++j) g[j] = std::exp((double)zt[sel[j]] - z0) / s;
            for (int j = 0; j < k; ++j) dot += g[j] * dgt[j];
            for (int j = 0; j < k; ++j) dz[(size_t)t * k + j] = g[j] * (dgt[j] - dot);
        } else if (D->gate_mode == 1) {
            std::vector<double> sg(k);
            double s = 0, dot = 0;
            for (int j = 0; j < k; ++j) { sg[j] = sigmoid(zt[sel[j]]); s += sg[j]; }
            for (int j = 0; j < k; ++j) dot += sg[j] / s * dgt[j];
            for (int j = 0; j < k; ++j) dz[(size_t)t * k + j] = (dgt[j] - dot) / s * sg[j] * (1.0 - sg[j]);
        } else if (D->gate_mode == 2) {
            std::vector<double> p(E);
            double m = zt[sel[0]], s = 0;
            for (int e = 0; e < E; ++e) s += std::exp((double)zt[e] - m);
            for (int e = 0; e < E; ++e) p[e] = std::exp((double)zt[e] - m) / s;
            for (int e = 0; e < E; ++e) {
                double v = 0;
                for (int j = 0; j < k; ++j) v += dgt[j] * p[sel[j]] * ((e == sel[j] ? 1.0 : 0.0) - p[e]);
                dz[(size_t)t * E + e] = v;
            }
        } else {
            return -4;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Scheduler oracle (c-sched).  PAPER.md §4.3.1: one queue per stream; the ready
// set = tasks whose upstream tasks are all scheduled; repeat { pick the ready task with the most
// downstream dependencies; append it to the queue of its stream; mark it scheduled }.
// Reading c-21: "downstream dependencies" = number of transitive descendants; ties -> lower
// `prio` value first (forward chunk before backward chunk), then lower node id.
// PAPER.md §4.3.2: a task waits on the event of every dependency that ran on a
// different stream; a task records an event iff some consumer runs on a different stream.
// Outputs: order[n] (pick sequence), n_desc[n], waits as pairs (producer, consumer) in
// (consumer pick order, producer id) order -> wait_pairs[2*n_waits], records[n] (0/1).
// ---------------------------------------------------------------------------------------------
int oracle_list_schedule(int32_t n, int32_t n_edges, const int32_t* edges /*[n_edges][2] src,dst*/,
                         const int32_t* stream_of, const int32_t* prio, int32_t* order, int32_t* n_desc,
                         int32_t* wait_pairs, int32_t* n_waits, int32_t* records) {
    std::vector<std::vector<int>> succ(n), pred(n);
    for (int i = 0; i < n_edges; ++i) {
        int s = edges[2 * i], t = edges[2 * i + 1];
        if (s < 0 || s >= n || t < 0 || t >= n || s == t) return -1;
        succ[s].push_back(t);
        pred[t].push_back(s);
    }
    // transitive descendant counts by depth-first reachability from every node
    for (int v = 0; v < n; ++v) {
        std::vector<char> seen(n, 0);
        std::vector<int> stack(1, v);
        int cnt = 0;
        while (!stack.empty()) {
            int a = stack.back();
            stack.pop_back();
            for (int b : succ[a])
                if (!seen[b]) { seen[b] = 1; ++cnt; stack.push_back(b); }
        }
        if (seen[v]) return -2;  // cycle
        n_desc[v] = cnt;
    }
    std::vector<char> done(n, 0);
    for (int step = 0; step < n; ++step) {
        int best = -1;
        for (int v = 0; v < n; ++v) {
            if (done[v]) continue;
            bool ready = true;
            for (int p : pred[v]) ready = ready && done[p];
            if (!ready) continue;
            if (best < 0 || n_desc[v] > n_desc[best] ||
                (n_desc[v] == n_desc[best] && prio[v] < prio[best]))
                best = v;  // equal desc and prio: the lower id, met first, stays
        }
        if (best < 0) return -2;
        done[best] = 1;
        order[step] = best;
    }
    int nw = 0;
    for (int v = 0; v < n; ++v) records[v] = 0;
    for (int step = 0; step < n; ++step) {
        int v = order[step];
        std::vector<int> ps(pred[v]);
        std::sort(ps.begin(), ps.end());
        for (int p : ps)
            if (stream_of[p] != stream_of[v]) {
                wait_pairs[2 * nw] = p;
                wait_pairs[2 * nw + 1] = v;
                ++nw;
                records[p] = 1;
            }
    }
    *n_waits = nw;
    return 0;
}

}  // extern "C"
