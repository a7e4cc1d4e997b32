// sched.cpp — host-only list scheduler of piper_run_chunk_pair (no CUDA in this file).
// PAPER.md §4.3.1 (lines 267-271): keep one queue per stream; repeatedly take, among the tasks whose
// upstream tasks are all scheduled, the one with the most downstream dependencies, append it to the
// queue of its stream and mark it scheduled.  Reading c-21: "downstream dependencies" =
// transitive descendants; ties go to the lower `prio`, then the lower task id (PAPER.md:290 asks for a
// deterministic order).  PAPER.md §4.3.2 (lines 279-286): a task waits on an event only for a
// dependency that ran on another stream, and records one only if a consumer runs on another stream.
#include <cstdint>
#include <utility>
#include <unordered_map>
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
// duration per task the static two-stream schedule of a DAG of this size can be searched exactly.  A schedule is a
// pair of per-stream sequences, run under the event rule (a task starts when its stream is free and all its
// producers have finished).  The search appends ready tasks depth first, task ids ascending, and cuts a branch
//  (a) whose lower bound - the remaining work of either stream, or the earliest start of a ready task plus the longest
//      chain behind it - cannot beat the best schedule found so far, or
//  (b) whose state is dominated by a state seen before with the same set of scheduled tasks: both streams free no
//      later and every producer that still has consumers finished no later (whatever completes the one completes the
//      other no later; this is what folds the orders of independent tasks into one).
// The first schedule with the smallest makespan in that order wins, so the result is a pure function of the inputs
// (PAPER.md:290).  A budget of kSearchNodes visited states bounds the host time on adversarial DAGs (the pair DAG with
// its four caller tasks takes ~10^3): past it the best schedule found so far is returned.
namespace {

constexpr long long kSearchNodes = 1 << 21;

struct Seen {
    double free_at[2];
    double fin[18];  // finish time of scheduled tasks that still have unscheduled consumers, else 0
};

struct Search {
    int n = 0;
    std::vector<std::vector<int32_t>> preds, succs;
    const int32_t* stream_of = nullptr;
    const float* dur = nullptr;
    std::vector<double> tail;  // dur[v] + the longest chain of successors behind v (streams ignored)
    std::vector<double> fin;
    std::vector<char> used;
    std::vector<int32_t> cur, best_order;
    std::unordered_map<uint32_t, Seen> seen;
    uint32_t mask = 0;
    long long nodes = 0;
    double free_at[2] = {0, 0}, rem[2] = {0, 0}, best = -1.0;

    double start_of(int32_t v) const {
        double start = free_at[stream_of[v]];
        for (int32_t p : preds[v])
            if (fin[p] > start) start = fin[p];
        return start;
    }
    bool ready(int32_t v) const {
        if (used[v]) return false;
        for (int32_t p : preds[v])
            if (!used[p]) return false;
        return true;
    }
    // true when a state seen before with this set of scheduled tasks is no later in every respect; records this one otherwise
    bool dominated() {
        Seen now;
        now.free_at[0] = free_at[0], now.free_at[1] = free_at[1];
        for (int32_t v = 0; v < 18; ++v) now.fin[v] = 0;
        for (int32_t v = 0; v < n; ++v) {
            if (!used[v]) continue;
            for (int32_t t : succs[v])
                if (!used[t]) now.fin[v] = fin[v];
        }
        auto it = seen.find(mask);
        if (it == seen.end()) {
            seen.emplace(mask, now);
            return false;
        }
        const Seen& old = it->second;
        bool old_le = old.free_at[0] <= now.free_at[0] + 1e-12 && old.free_at[1] <= now.free_at[1] + 1e-12;
        bool now_le = now.free_at[0] <= old.free_at[0] + 1e-12 && now.free_at[1] <= old.free_at[1] + 1e-12;
        for (int32_t v = 0; v < n; ++v) {
            old_le = old_le && old.fin[v] <= now.fin[v] + 1e-12;
            now_le = now_le && now.fin[v] <= old.fin[v] + 1e-12;
        }
        if (old_le) return true;
        if (now_le) it->second = now;  // the better of two comparable states is kept; incomparable: the first
        return false;
    }
    void dfs() {
        if ((int)cur.size() == n) {
            const double m = free_at[0] > free_at[1] ? free_at[0] : free_at[1];
            if (best < 0 || m < best - 1e-9) best = m, best_order = cur;
            return;
        }
        if (best >= 0 && ++nodes > kSearchNodes) return;  // budget spent: keep the best schedule found
        double lb = free_at[0] + rem[0] > free_at[1] + rem[1] ? free_at[0] + rem[0] : free_at[1] + rem[1];
        for (int32_t v = 0; v < n; ++v)
            if (ready(v)) {
                const double e = start_of(v) + tail[v];
                if (e > lb) lb = e;
            }
        if (best >= 0 && lb >= best - 1e-9) return;
        if (!cur.empty() && dominated()) return;
        for (int32_t v = 0; v < n; ++v) {
            if (!ready(v)) continue;
            const double start = start_of(v);
            const int s = stream_of[v];
            const double keep_free = free_at[s];
            used[v] = 1, mask |= 1u << v, fin[v] = start + dur[v], free_at[s] = fin[v], rem[s] -= dur[v], cur.push_back(v);
            dfs();
            cur.pop_back(), rem[s] += dur[v], free_at[s] = keep_free, fin[v] = -1.0, mask &= ~(1u << v), used[v] = 0;
        }
    }
};

}  // namespace

extern "C" int piper_schedule_search(int32_t n, int32_t n_edges, const int32_t* edges, const int32_t* stream_of,
                                     const float* dur, int32_t* order, int32_t* waits, int32_t* n_waits,
                                     int32_t* records, float* makespan) {
    if (n < 0 || n > 18 || n_edges < 0 || (n_edges > 0 && !edges) || (n > 0 && (!stream_of || !dur || !order || !records)) ||
        !n_waits)
        return PIPER_ERR_INVALID;
    Search S;
    S.n = n, S.stream_of = stream_of, S.dur = dur;
    S.preds.assign(n, {});
    std::vector<std::vector<int32_t>>& succs = S.succs;
    succs.assign(n, {});
    for (int32_t i = 0; i < n_edges; ++i) {
        const int32_t s = edges[2 * i], t = edges[2 * i + 1];
        if (s < 0 || s >= n || t < 0 || t >= n || s == t) return PIPER_ERR_INVALID;
        S.preds[t].push_back(s), succs[s].push_back(t);
    }
    for (int32_t v = 0; v < n; ++v)
        if ((stream_of[v] != 0 && stream_of[v] != 1) || !(dur[v] >= 0.f)) return PIPER_ERR_INVALID;
    // longest chain behind every task, in reverse topological order (Kahn on the successor counts); a cycle leaves tasks out
    S.tail.assign(n, 0.0);
    {
        std::vector<int32_t> left(n), stack;
        for (int32_t v = 0; v < n; ++v) {
            left[v] = (int32_t)succs[v].size();
            if (!left[v]) stack.push_back(v);
        }
        int32_t done = 0;
        while (!stack.empty()) {
            const int32_t v = stack.back();
            stack.pop_back(), ++done;
            double longest = 0;
            for (int32_t t : succs[v])
                if (S.tail[t] > longest) longest = S.tail[t];
            S.tail[v] = dur[v] + longest;
            for (int32_t p : S.preds[v])
                if (--left[p] == 0) stack.push_back(p);
        }
        if (done != n) return PIPER_ERR_INVALID;  // cycle
    }
    S.fin.assign(n, -1.0), S.used.assign(n, 0);
    for (int32_t v = 0; v < n; ++v) S.rem[stream_of[v]] += dur[v];
    S.dfs();
    const double best = S.best;
    const std::vector<int32_t>& best_order = S.best_order;
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
