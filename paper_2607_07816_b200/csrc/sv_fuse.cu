// Host-side gate fusion: "for each block of single- and two-qubit gates we
// fuse those gates into a multi-qubit unitary operation ... one update per block", and truncation then runs once
// per block.  Blocks are formed greedily over CONSECUTIVE gates: a gate joins the running block while the union of
// qubits stays within max_m, otherwise the block is closed and the gate opens the next one.  The fused unitary is
// fed to the same hot path (sv_apply_gate / sv_apply_gate_truncate), whose classification by zero pattern then
// sees what the product really mixes (a diagonal times a CNOT is still a monomial one-bit gate).
// Host code only: no kernel, no device memory.
#include <string.h>

#include <vector>

#include "../../include/sparse_sv.h"

namespace {
struct Cx { double re, im; };
inline Cx cmul(Cx a, Cx b) { return Cx{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }

struct Block {
    int m = 0;
    int q[SV_FUSE_MAX_M];
    std::vector<Cx> U;   // 2^m x 2^m, row-major; local bit j <-> q[j]
};

// U <- U (x) I on one more (most significant) local bit
void grow(Block& b, int qubit) {
    const int d = 1 << b.m, D = d << 1;
    std::vector<Cx> V((size_t)D * D, Cx{0.0, 0.0});
    for (int r = 0; r < d; ++r)
        for (int c = 0; c < d; ++c) {
            V[(size_t)r * D + c] = b.U[(size_t)r * d + c];
            V[(size_t)(r + d) * D + (c + d)] = b.U[(size_t)r * d + c];
        }
    b.U.swap(V);
    b.q[b.m++] = qubit;
}

// U <- E(G) U, E(G) = the gate G (on local positions pos[0..mg-1] of the block) embedded in the block's space
void absorb(Block& b, const Cx* G, int mg, const int* pos) {
    const int D = 1 << b.m, dg = 1 << mg;
    int gmask = 0;
    for (int i = 0; i < mg; ++i) gmask |= 1 << pos[i];
    std::vector<Cx> V((size_t)D * D);
    for (int r = 0; r < D; ++r) {
        int gr = 0;
        for (int i = 0; i < mg; ++i) gr |= ((r >> pos[i]) & 1) << i;
        const int rest = r & ~gmask;
        for (int c = 0; c < D; ++c) {
            Cx s{0.0, 0.0};
            for (int gc = 0; gc < dg; ++gc) {          // ascending column index of the gate
                int k = rest;
                for (int i = 0; i < mg; ++i) k |= ((gc >> i) & 1) << pos[i];
                const Cx t = cmul(G[gr * dg + gc], b.U[(size_t)k * D + c]);
                s.re += t.re; s.im += t.im;
            }
            V[(size_t)r * D + c] = s;
        }
    }
    b.U.swap(V);
}

int fuse_impl(int n_gates, const int* gate_m, const int* gate_qubits, const sv_c128* gate_U, int max_m,
                             int* n_blocks, int* block_m, int* block_qubits, sv_c128* block_U, size_t block_U_capacity) {
    if (n_gates < 0 || max_m < 1 || max_m > SV_FUSE_MAX_M || !n_blocks || (n_gates && (!gate_m || !gate_qubits || !gate_U)) ||
        (n_gates && (!block_m || !block_qubits || !block_U)))
        return SV_ERR_INVALID_ARG;
    *n_blocks = 0;
    size_t qoff = 0, uoff = 0, out_q = 0, out_u = 0;
    Block b;
    auto flush = [&]() -> int {
        if (b.m == 0) return SV_OK;
        const size_t need = (size_t)1 << (2 * b.m);
        if (out_u + need > block_U_capacity) return SV_ERR_INVALID_ARG;
        block_m[*n_blocks] = b.m;
        for (int j = 0; j < b.m; ++j) block_qubits[out_q + j] = b.q[j];
        memcpy(block_U + out_u, b.U.data(), need * sizeof(sv_c128));
        out_q += b.m; out_u += need; *n_blocks += 1;
        b.m = 0; b.U.clear();
        return SV_OK;
    };
    for (int g = 0; g < n_gates; ++g) {
        const int mg = gate_m[g];
        if (mg < 1 || mg > max_m) return SV_ERR_INVALID_ARG;
        const int* q = gate_qubits + qoff;
        for (int i = 0; i < mg; ++i) {
            if (q[i] < 0 || q[i] >= 64) return SV_ERR_INVALID_ARG;
            for (int j = 0; j < i; ++j) if (q[j] == q[i]) return SV_ERR_INVALID_ARG;
        }
        int fresh = 0;
        for (int i = 0; i < mg; ++i) {
            bool in = false;
            for (int j = 0; j < b.m; ++j) in = in || b.q[j] == q[i];
            fresh += in ? 0 : 1;
        }
        if (b.m + fresh > max_m) { const int rc = flush(); if (rc != SV_OK) return rc; }
        if (b.m == 0) b.U.assign(1, Cx{1.0, 0.0});
        int pos[SV_FUSE_MAX_M];
        for (int i = 0; i < mg; ++i) {
            int p = -1;
            for (int j = 0; j < b.m; ++j) if (b.q[j] == q[i]) p = j;
            if (p < 0) { grow(b, q[i]); p = b.m - 1; }
            pos[i] = p;
        }
        absorb(b, reinterpret_cast<const Cx*>(gate_U + uoff), mg, pos);
        qoff += mg; uoff += (size_t)1 << (2 * mg);
    }
    return flush();
}
}  // namespace

// (std::vector may throw: no C++ exception crosses the C ABI)
extern "C" int sv_fuse_gates(int n_gates, const int* gate_m, const int* gate_qubits, const sv_c128* gate_U, int max_m,
                             int* n_blocks, int* block_m, int* block_qubits, sv_c128* block_U, size_t block_U_capacity) {
    try {
        return fuse_impl(n_gates, gate_m, gate_qubits, gate_U, max_m, n_blocks, block_m, block_qubits, block_U, block_U_capacity);
    } catch (...) {
        return SV_ERR_NOMEM;
    }
}
