// sched.cpp — host-only list scheduler of piper_run_chunk_pair (no CUDA in this file).
// PAPER.md §4.3.1 (lines 267-271): keep one queue per stream; repeatedly take, among the tasks whose
// upstream tasks are all scheduled, the one with the most downstream dependencies, append it to the
// queue of its stream and mark it scheduled.  Reading c-21: "downstream dependencies" =
// transitive descendants; ties go to the lower `prio`, then the lower task id (PAPER.md:290 asks for a
// deterministic order).  PAPER.md §4.3.2 (lines 279-286): a task waits on an event only for a
// dependency that ran on another stream, and records one only if a consumer runs on another stream.
#include <cstdint>
#include <utility>
#include <vector>

#include "piper.h"

extern "C" int piper_list_schedule(int32_t n, int32_t n_edges, const int32_t* edges, const int32_t* stream_of,
                                   const int32_t* prio, int32_t* order, int32_t* waits, int32_t* n_waits,
                                   int32_t* records) {
    if (n < 0 || n_edges < 0 || (n_edges > 0 && !edges) || (n > 0 && (!stream_of || !prio || !order || !records)) ||
        !n_waits)
        return PIPER_ERR_INVALID;
    for (int32_t i = 0; i < n_edges; ++i) {
        const int32_t s = edges[2 * i], t = edges[2 * i + 1];
        if (s < 0 || s >= n || t < 0 || t >= n || s == t) return PIPER_ERR_INVALID;
    }
    // reach[v] = bitset of descendants, filled in reverse topological order (Kahn)
    std::vector<int32_t> indeg(n, 0), topo;
    for (int32_t i = 0; i < n_edges; ++i) indeg[edges[2 * i + 1]] += 1;
    for (int32_t v = 0; v < n; ++v)
        if (indeg[v] == 0) topo.push_back(v);
    for (size_t h = 0; h < topo.size(); ++h)
        for (int32_t i = 0; i < n_edges; ++i)
            if (edges[2 * i] == topo[h] && --indeg[edges[2 * i + 1]] == 0) topo.push_back(edges[2 * i + 1]);
    if ((int32_t)topo.size() != n) return PIPER_ERR_INVALID;  // cycle
    const int words = (n + 63) / 64;
    std::vector<uint64_t> reach((size_t)n * words, 0);
    for (int32_t h = n - 1; h >= 0; --h) {
        const int32_t v = topo[h];
        for (int32_t i = 0; i < n_edges; ++i)
            if (edges[2 * i] == v) {
                const int32_t t = edges[2 * i + 1];
                reach[(size_t)v * words + t / 64] |= 1ull << (t % 64);
                for (int w = 0; w < words; ++w) reach[(size_t)v * words + w] |= reach[(size_t)t * words + w];
            }
    }
    std::vector<int32_t> ndesc(n, 0), pending(n, 0);
    for (int32_t v = 0; v < n; ++v)
        for (int w = 0; w < words; ++w) ndesc[v] += __builtin_popcountll(reach[(size_t)v * words + w]);
    for (int32_t i = 0; i < n_edges; ++i) pending[edges[2 * i + 1]] += 1;
    std::vector<char> scheduled(n, 0);
    for (int32_t step = 0; step < n; ++step) {
        int32_t pick = -1;
        for (int32_t v = 0; v < n; ++v) {
            if (scheduled[v] || pending[v] != 0) continue;
            if (pick < 0 || ndesc[v] > ndesc[pick] || (ndesc[v] == ndesc[pick] && prio[v] < prio[pick])) pick = v;
        }
        scheduled[pick] = 1;
        order[step] = pick;
        for (int32_t i = 0; i < n_edges; ++i)
            if (edges[2 * i] == pick) pending[edges[2 * i + 1]] -= 1;
    }
    int32_t nw = 0;
    for (int32_t v = 0; v < n; ++v) records[v] = 0;
    for (int32_t step = 0; step < n; ++step) {
        const int32_t v = order[step];
        for (int32_t p = 0; p < n; ++p) {  // producers in ascending id
            bool is_pred = false;
            for (int32_t i = 0; i < n_edges; ++i) is_pred = is_pred || (edges[2 * i] == p && edges[2 * i + 1] == v);
            if (is_pred && stream_of[p] != stream_of[v]) {
                if (waits) waits[2 * nw] = p, waits[2 * nw + 1] = v;
                ++nw;
                records[p] = 1;
            }
        }
    }
    *n_waits = nw;
    return PIPER_OK;
}

// ---- profile-guided variant ---------------------------------------------------------------------------
// PAPER.md:273 and 420 name profile-guided scheduling as the way past the simple policy above.  With a
// duration per task the static two-stream schedule can be searched exhaustively for a DAG of this size:
// every pair of per-stream sequences (linear extensions of the DAG restricted to a stream) is simulated
// under the event rule (a task starts when its stream is free and all its producers have finished) and
// the pair with the smallest makespan wins; ties go to the lexicographically smallest pick sequence, so
// the result is a pure function of the inputs.
namespace {

struct Search {
    int n;
    std::vector<std::vector<int32_t>> preds;
    const int32_t* stream_of;
    const float* dur;
    std::vector<std::vector<int32_t>> seqs[2];

    void extensions(int s, std::vector<int32_t>& cur, std::vector<char>& used) {
        bool any = false;
        for (int32_t v = 0; v < n; ++v) {
            if (stream_of[v] != s || used[v]) continue;
            bool ok = true;
            for (int32_t p : preds[v]) ok = ok && (stream_of[p] != s || used[p]);
            if (!ok) continue;
            any = true;
            used[v] = 1, cur.push_back(v);
            extensions(s, cur, used);
            cur.pop_back(), used[v] = 0;
        }
        if (!any) {
            size_t want = 0;
            for (int32_t v = 0; v < n; ++v) want += stream_of[v] == s;
            if (cur.size() == want) seqs[s].push_back(cur);
        }
    }
    // simulate; returns makespan or a negative value on deadlock; `order` = tasks by start time
    double simulate(const std::vector<int32_t>& a, const std::vector<int32_t>& b, std::vector<int32_t>& order) const {
        const std::vector<int32_t>* q[2] = {&a, &b};
        size_t head[2] = {0, 0};
        double free_at[2] = {0, 0};
        std::vector<double> fin(n, -1.0);
        order.clear();
        while (head[0] < a.size() || head[1] < b.size()) {
            int pick = -1;
            double best = 0;
            for (int s = 0; s < 2; ++s) {
                if (head[s] >= q[s]->size()) continue;
                const int32_t v = (*q[s])[head[s]];
                double start = free_at[s];
                bool ready = true;
                for (int32_t p : preds[v]) {
                    if (fin[p] < 0) ready = false;
                    else if (fin[p] > start) start = fin[p];
                }
                if (ready && (pick < 0 || start < best)) pick = s, best = start;
            }
            if (pick < 0) return -1.0;
            const int32_t v = (*q[pick])[head[pick]++];
            fin[v] = best + dur[v], free_at[pick] = fin[v];
            order.push_back(v);
        }
        return free_at[0] > free_at[1] ? free_at[0] : free_at[1];
    }
};

}  // namespace

extern "C" int piper_schedule_search(int32_t n, int32_t n_edges, const int32_t* edges, const int32_t* stream_of,
                                     const float* dur, int32_t* order, int32_t* waits, int32_t* n_waits,
                                     int32_t* records, float* makespan) {
    if (n < 0 || n > 16 || n_edges < 0 || (n_edges > 0 && !edges) || (n > 0 && (!stream_of || !dur || !order || !records)) ||
        !n_waits)
        return PIPER_ERR_INVALID;
    Search S;
    S.n = n, S.stream_of = stream_of, S.dur = dur;
    S.preds.assign(n, {});
    for (int32_t i = 0; i < n_edges; ++i) {
        const int32_t s = edges[2 * i], t = edges[2 * i + 1];
        if (s < 0 || s >= n || t < 0 || t >= n || s == t) return PIPER_ERR_INVALID;
        S.preds[t].push_back(s);
    }
    for (int32_t v = 0; v < n; ++v)
        if ((stream_of[v] != 0 && stream_of[v] != 1) || !(dur[v] >= 0.f)) return PIPER_ERR_INVALID;
    for (int s = 0; s < 2; ++s) {
        std::vector<int32_t> cur;
        std::vector<char> used(n, 0);
        S.extensions(s, cur, used);
    }
    double best = -1.0;
    std::vector<int32_t> best_order, cand;
    for (const auto& a : S.seqs[0])
        for (const auto& b : S.seqs[1]) {
            const double m = S.simulate(a, b, cand);
            if (m < 0) continue;
            if (best < 0 || m < best - 1e-9 || (m < best + 1e-9 && cand < best_order)) best = m, best_order = cand;
        }
    if (best < 0) return PIPER_ERR_INVALID;  // cycle
    for (int32_t i = 0; i < n; ++i) order[i] = best_order[i];
    int32_t nw = 0;
    for (int32_t v = 0; v < n; ++v) records[v] = 0;
    for (int32_t step = 0; step < n; ++step) {
        const int32_t v = order[step];
        std::vector<int32_t> ps = S.preds[v];
        for (size_t i = 0; i < ps.size(); ++i)  // producers in ascending id, each once
            for (size_t j = i + 1; j < ps.size(); ++j)
                if (ps[j] < ps[i]) std::swap(ps[i], ps[j]);
        for (size_t i = 0; i < ps.size(); ++i) {
            if (i > 0 && ps[i] == ps[i - 1]) continue;
            if (stream_of[ps[i]] != stream_of[v]) {
                if (waits) waits[2 * nw] = ps[i], waits[2 * nw + 1] = v;
                ++nw;
                records[ps[i]] = 1;
            }
        }
    }
    *n_waits = nw;
    if (makespan) *makespan = (float)best;
    return PIPER_OK;
}
