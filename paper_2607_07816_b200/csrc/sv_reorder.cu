// Host-side gate reordering: "we reorder the gates so that, during simulation, the
// set of currently active qubits is kept as small as possible, while the introduction of additional qubits is
// postponed for as long as the circuit dependencies allow ... we only reorder commuting gates or dependency-compatible
// gates".  The paper gives no algorithm; the reading taken (R20) is a greedy list schedule:
//   * two gates CONFLICT when they share a qubit, unless both are flagged diagonal (diagonal gates commute);
//   * a gate is READY when every earlier gate it conflicts with has been scheduled (so the relative order of every
//     conflicting pair is kept and the reordered circuit is the same operator);
//   * a qubit is ACTIVE once a scheduled gate has touched it;
//   * each step schedules the ready gate that activates the fewest new qubits, ties to the lowest original index.
// Host code only: no kernel, no device memory.  O(n_gates^2) for the dependency lists, which is nothing beside one pass
// over a state.
#include <stdint.h>

#include <vector>

#include "../../include/sparse_sv.h"

static int reorder_impl(int n_gates, const int* gate_m, const int* gate_qubits, const unsigned char* gate_diag,
                        int* order, int* n_active_after) {
    if (n_gates < 0 || (n_gates && (!gate_m || !gate_qubits || !order))) return SV_ERR_INVALID_ARG;
    std::vector<uint64_t> qmask((size_t)n_gates, 0);
    {
        size_t off = 0;
        for (int g = 0; g < n_gates; ++g) {
            const int m = gate_m[g];
            if (m < 1 || m > 64) return SV_ERR_INVALID_ARG;
            for (int i = 0; i < m; ++i) {
                const int q = gate_qubits[off + i];
                if (q < 0 || q >= 64 || ((qmask[g] >> q) & 1)) return SV_ERR_INVALID_ARG;
                qmask[g] |= (uint64_t)1 << q;
            }
            off += m;
        }
    }
    // per qubit: the last non-diagonal gate seen and the diagonal gates since (they commute with one another)
    std::vector<int> last_nd(64, -1);
    std::vector<std::vector<int>> diags_since(64);
    std::vector<std::vector<int>> succ((size_t)n_gates);
    std::vector<int> waiting((size_t)n_gates, 0);
    auto edge = [&](int from, int to) { succ[(size_t)from].push_back(to); ++waiting[(size_t)to]; };
    for (int g = 0; g < n_gates; ++g) {
        const bool dg = gate_diag && gate_diag[g];
        for (int q = 0; q < 64; ++q) {
            if (!((qmask[g] >> q) & 1)) continue;
            if (last_nd[q] >= 0) edge(last_nd[q], g);
            if (dg) {
                diags_since[q].push_back(g);
            } else {
                for (int d : diags_since[q]) edge(d, g);
                diags_since[q].clear();
                last_nd[q] = g;
            }
        }
    }
    std::vector<char> done((size_t)n_gates, 0);
    uint64_t active = 0;
    for (int step = 0; step < n_gates; ++step) {
        int best = -1, best_new = 65;
        for (int g = 0; g < n_gates; ++g) {
            if (done[g] || waiting[g]) continue;
            const int fresh = __builtin_popcountll(qmask[g] & ~active);
            if (fresh < best_new) { best = g; best_new = fresh; if (fresh == 0) break; }
        }
        if (best < 0) return SV_ERR_INVALID_ARG;   // cannot happen: the conflict relation only points forward
        done[best] = 1;
        active |= qmask[best];
        for (int t : succ[(size_t)best]) --waiting[(size_t)t];
        order[step] = best;
        if (n_active_after) n_active_after[step] = __builtin_popcountll(active);
    }
    return SV_OK;
}

// (std::vector may throw: no C++ exception crosses the C ABI)
extern "C" int sv_reorder_gates(int n_gates, const int* gate_m, const int* gate_qubits, const unsigned char* gate_diag,
                                int* order, int* n_active_after) {
    try {
        return reorder_impl(n_gates, gate_m, gate_qubits, gate_diag, order, n_active_after);
    } catch (...) {
        return SV_ERR_NOMEM;
    }
}
