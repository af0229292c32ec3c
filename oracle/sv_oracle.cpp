// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, single-threaded sparse state-vector simulator written from the paper
// (arxiv/paper_2607_07816, /root/reference/PAPER.md).  It is the parity reference and the
// timed "cpu_baseline" of bench.py.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.  It shares no code, header, table or
// helper with the CUDA engine under paper_2607_07816_b200/csrc/.
//
// State: std::unordered_map<uint64 basis index -> complex128 amplitude>, nonzero terms
// only.
//
//   orc_apply_gate  the sparse form of Eq. 3 generalised to m qubits (PAPER.md:47, :49,
//                   :110-118): every tuple of 2^m amplitudes whose basis states differ only
//                   in the gate's qubits is multiplied by U; absent amplitudes are 0;
//                   results that are exactly 0+0i are not stored.  [pinned: dense 2^n
//                   simulator, closed forms -- tests/test_oracle_*.py]
//   orc_truncate    PAPER.md:94-96, :124: sort by |a|^2 descending (ties: key ascending,
//                   DESIGN.md reading R4), p-mass prefix first, then top-k, then
//                   renormalise once (R6); a call that drops nothing leaves the state
//                   bitwise untouched (R7).  [pinned: closed forms + numpy lexsort brute force]
//   orc_norm        sum |a|^2 (Eq. 4)
//   orc_top         the k most probable terms in (p desc, key asc) order
//
// Arithmetic contract: complex product written out as
// (ur*ar - ui*ai, ur*ai + ui*ar), contributions added in ascending local column index c,
// every operation rounded separately (build with -ffp-contract=off), p = re*re + im*im.
//
// Conventions: qubit q = bit q of the key (R1); local index bit j = key bit qubits[j];
// U row-major U[r*2^m + c] (R2).

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <unordered_map>
#include <unordered_set>
#include <vector>

namespace {

typedef std::complex<double> cplx;

struct Oracle {
    int n;
    std::unordered_map<uint64_t, cplx> terms;
};

struct Rec {
    double p;
    uint64_t key;
    cplx a;
};

inline bool rec_less(const Rec& x, const Rec& y) {  // (p desc, key asc)  [R4]
    if (x.p != y.p) return x.p > y.p;
    return x.key < y.key;
}

inline uint64_t scatter_bits(unsigned c, const int* qubits, int m) {
    uint64_t s = 0;
    for (int j = 0; j < m; ++j)
        if ((c >> j) & 1u) s |= (uint64_t)1 << qubits[j];
    return s;
}

std::vector<Rec> sorted_records(const Oracle* o) {
    std::vector<Rec> v;
    v.reserve(o->terms.size());
    for (const auto& kv : o->terms) {
        double re = kv.second.real(), im = kv.second.imag();
        double p = re * re + im * im;  // two products, one sum, no FMA
        v.push_back(Rec{p, kv.first, kv.second});
    }
    std::sort(v.begin(), v.end(), rec_less);
    return v;
}

}  // namespace

extern "C" {

void* orc_create(int n_qubits) {
    if (n_qubits < 1 || n_qubits > 64) return nullptr;
    Oracle* o = new Oracle();
    o->n = n_qubits;
    o->terms[0] = cplx(1.0, 0.0);  // ground state |0...0>
    return o;
}

void orc_destroy(void* h) { delete static_cast<Oracle*>(h); }

uint64_t orc_num_terms(void* h) { return static_cast<Oracle*>(h)->terms.size(); }

// Replace the state by the given terms (keys must be distinct; zero amplitudes are skipped).
int orc_load(void* h, const uint64_t* keys, const double* amps, uint64_t count) {
    Oracle* o = static_cast<Oracle*>(h);
    std::unordered_map<uint64_t, cplx> t;
    t.reserve(count * 2);
    for (uint64_t i = 0; i < count; ++i) {
        if (o->n < 64 && (keys[i] >> o->n) != 0) return -1;
        cplx a(amps[2 * i], amps[2 * i + 1]);
        if (a.real() == 0.0 && a.imag() == 0.0) continue;
        if (!t.emplace(keys[i], a).second) return -1;
    }
    o->terms.swap(t);
    return 0;
}

// PAPER.md:110-118.  U: 2^m x 2^m row-major, interleaved (re, im).
int orc_apply_gate(void* h, const int* qubits, int m, const double* U) {
    Oracle* o = static_cast<Oracle*>(h);
    if (m < 1 || m > 6) return -1;
    uint64_t mask = 0;
    for (int j = 0; j < m; ++j) {
        if (qubits[j] < 0 || qubits[j] >= o->n) return -1;
        uint64_t b = (uint64_t)1 << qubits[j];
        if (mask & b) return -1;
        mask |= b;
    }
    const unsigned d = 1u << m;
    std::unordered_map<uint64_t, cplx> out;
    out.reserve(o->terms.size() * 2);
    std::unordered_set<uint64_t> done;
    done.reserve(o->terms.size() * 2);
    std::vector<cplx> a(d);
    for (const auto& kv : o->terms) {
        const uint64_t base = kv.first & ~mask;        // equal pattern in the remaining qubits
        if (!done.insert(base).second) continue;       // each tuple exactly once
        for (unsigned c = 0; c < d; ++c) {             // the 2^m-tuple; absent = 0
            auto it = o->terms.find(base | scatter_bits(c, qubits, m));
            a[c] = (it == o->terms.end()) ? cplx(0.0, 0.0) : it->second;
        }
        for (unsigned r = 0; r < d; ++r) {             // column c times amplitude c, summed
            double sr = 0.0, si = 0.0;
            for (unsigned c = 0; c < d; ++c) {
                const double ur = U[2 * (r * d + c)], ui = U[2 * (r * d + c) + 1];
                const double ar = a[c].real(), ai = a[c].imag();
                const double pr = ur * ar - ui * ai;
                const double pi = ur * ai + ui * ar;
                sr = sr + pr;
                si = si + pi;
            }
            if (sr == 0.0 && si == 0.0) continue;      // only nonzero amplitudes are stored
            out.emplace(base | scatter_bits(r, qubits, m), cplx(sr, si));
        }
    }
    o->terms.swap(out);
    return 0;
}

double orc_norm(void* h) {
    Oracle* o = static_cast<Oracle*>(h);
    std::vector<Rec> v = sorted_records(o);
    double s = 0.0;
    for (const Rec& r : v) s = s + r.p;
    return s;
}

// PAPER.md:94-96, :124.  max_terms == 0: no cap.  min_mass >= 1: no mass threshold.
int orc_truncate(void* h, uint64_t max_terms, double min_mass, double* kept_fraction) {
    Oracle* o = static_cast<Oracle*>(h);
    if (!(min_mass > 0.0)) return -1;
    std::vector<Rec> v = sorted_records(o);              // sort from largest to smallest probability
    const uint64_t count = v.size();
    double S = 0.0;
    for (const Rec& r : v) S = S + r.p;
    uint64_t j_mass = count;
    if (min_mass < 1.0) {                                // p-mass first: smallest prefix with cum >= min_mass * S  [R5]
        const double thr = min_mass * S;
        double cum = 0.0;
        for (uint64_t i = 0; i < count; ++i) {
            cum = cum + v[i].p;
            if (cum >= thr) { j_mass = i + 1; break; }
        }
    }
    uint64_t j = j_mass;
    if (max_terms != 0 && max_terms < j) j = max_terms;  // then top-k
    if (j < 1 && count > 0) j = 1;
    if (j >= count) {                                    // nothing dropped: bitwise no-op  [R7]
        if (kept_fraction) *kept_fraction = 1.0;
        return 0;
    }
    double kept = 0.0;
    for (uint64_t i = 0; i < j; ++i) kept = kept + v[i].p;
    const double scale = 1.0 / std::sqrt(kept);          // renormalise once  [R6]
    std::unordered_map<uint64_t, cplx> out;
    out.reserve(j * 2);
    for (uint64_t i = 0; i < j; ++i)
        out.emplace(v[i].key, cplx(v[i].a.real() * scale, v[i].a.imag() * scale));
    o->terms.swap(out);
    if (kept_fraction) *kept_fraction = kept / S;
    return 0;
}

// The k most probable terms, (p desc, key asc).  Any output pointer may be null.
uint64_t orc_top(void* h, uint64_t k, uint64_t* keys, double* amps, double* probs) {
    Oracle* o = static_cast<Oracle*>(h);
    std::vector<Rec> v = sorted_records(o);
    const uint64_t w = std::min<uint64_t>(k, v.size());
    for (uint64_t i = 0; i < w; ++i) {
        if (keys) keys[i] = v[i].key;
        if (amps) { amps[2 * i] = v[i].a.real(); amps[2 * i + 1] = v[i].a.imag(); }
        if (probs) probs[i] = v[i].p;
    }
    return w;
}

}  // extern "C"
