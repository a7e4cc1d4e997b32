// sched.cpp — host-only list scheduler of piper_run_chunk_pair (no CUDA in this file).
// PAPER.md §4.3.1 (lines 267-271): keep one queue per stream; repeatedly take, among the tasks whose
// upstream tasks are all scheduled, the one with the most downstream dependencies, append it to the
// queue of its stream and mark it scheduled.  Reading c-21: "downstream dependencies" =
// transitive descendants; ties go to the lower `prio`, then the lower task id (PAPER.md:290 asks for a
// deterministic order).  PAPER.md §4.3.2 (lines 279-286): a task waits on an event only for a
// dependency that ran on another stream, and records one only if a consumer runs on another stream.
#include <cstdint>
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
