// Gate application kernels (SURVEY.md rows a-2 .. a-7).
//
// Storage invariant: keys are stored in a permuted ("physical") bit order and kept
// strictly ascending.  A gate never sorts: the qubits on which U actually mixes amplitudes
// ("active" bits) are moved to the least-significant physical positions one at a time,
// each move being ONE streaming pass -- a segmented two-way merge of the bit=0 run and the
// bit=1 run of every block of keys that agree above the moved bit.  After the last move
// the <= 2^ma terms of a tuple are adjacent, so the same pass forms the
// tuple, multiplies by U, drops exact zeros and writes unique, sorted keys (rows a-4..a-7
// fused).  Diagonal gates (row a-2) touch amplitudes only.
#include "sv_device.cuh"

// ---------------------------------------------------------------------------------------
// a-2 diagonal fast path: a <- U[c,c] * a, c = the key's pattern on the gate's qubits
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SV_THREADS) diag_kernel(const u64* __restrict__ keys, double2* __restrict__ amps,
                                                          u64 n, const GateTab* __restrict__ tab) {
    __shared__ double2 d[16];
    __shared__ int cpos[SV_MAX_M];
    __shared__ int mc_s;
    if (threadIdx.x < 16) d[threadIdx.x] = tab->U[threadIdx.x];
    if (threadIdx.x < SV_MAX_M) cpos[threadIdx.x] = tab->ctrl_pos[threadIdx.x];
    if (threadIdx.x == 0) mc_s = tab->mc;
    __syncthreads();
    const int mc = mc_s;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 k = ld_stream_u64(keys + i);
        double2 a = amps[i];
        int cx = 0;
        for (int j = 0; j < mc; ++j) cx |= (int)((k >> cpos[j]) & 1ull) << j;
        const double2 u = d[cx];
        double2 o;
        o.x = __dsub_rn(__dmul_rn(u.x, a.x), __dmul_rn(u.y, a.y));
        o.y = __dadd_rn(__dmul_rn(u.x, a.y), __dmul_rn(u.y, a.x));
        amps[i] = o;
    }
}

int svk_diag(const u64* keys, double2* amps, u64 n, const GateTab* tab, cudaStream_t st) {
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > 148ull * 16) blocks = 148ull * 16;
    diag_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, tab);
    return 1;
}

// ---------------------------------------------------------------------------------------
// tile boundaries of a bit-move pass (merge-path splits, one thread per boundary)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ u64 lower_bound_g(const u64* __restrict__ keys, u64 lo, u64 hi, u64 v) {
    while (lo < hi) {
        u64 mid = lo + ((hi - lo) >> 1);
        if (keys[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void find_splits_kernel(const u64* __restrict__ keys, u64 n, int p, int w, u32 tnom, u32 ntiles,
                                   TileDesc* __restrict__ desc) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > ntiles) return;
    const bool last = (j == ntiles);
    const u64 t = last ? n - 1 : (u64)j * tnom;   // n >= 1 here
    const u64 lowmask = (1ull << p) - 1;
    const u64 kt = keys[t];
    const u64 blk = (p == 63) ? 0 : ((kt >> (p + 1)) << (p + 1));
    const u64 s = (p == 63) ? 0 : lower_bound_g(keys, 0, t + 1, blk);
    const u64 mid = lower_bound_g(keys, s, n, blk | (1ull << p));
    u64 e = n;
    if (p < 63) {
        const u64 nxt = blk + (2ull << p);
        if (nxt != 0) e = lower_bound_g(keys, mid, n, nxt);   // nxt == 0: wrapped, last block
    }
    TileDesc d;
    d.mid = mid; d.e = e;
    if (last) { d.ia = mid; d.ib = e; desc[j] = d; return; }
    const u64 lenA = mid - s, lenB = e - mid, diag = t - s;
    u64 lo = diag > lenB ? diag - lenB : 0, hi = diag < lenA ? diag : lenA;
    while (lo < hi) {   // A first on ties: A[i] precedes B[diag-1-i] iff lowA <= lowB
        const u64 i = lo + ((hi - lo) >> 1);
        const u64 ka = keys[s + i] & lowmask, kb = keys[mid + (diag - 1 - i)] & lowmask;
        if (ka <= kb) lo = i + 1; else hi = i;
    }
    u64 i = lo, jb = diag - lo;
    if (w >= 0 && (i < lenA || jb < lenB)) {   // do not split a tuple: pull its earlier members across
        u64 nxt;
        if (i < lenA && jb < lenB) {
            const u64 ka = keys[s + i] & lowmask, kb = keys[mid + jb] & lowmask;
            nxt = ka <= kb ? ka : kb;
        } else nxt = (i < lenA) ? (keys[s + i] & lowmask) : (keys[mid + jb] & lowmask);
        const u64 v = nxt >> w;
        while (i > 0 && ((keys[s + i - 1] & lowmask) >> w) == v) --i;
        while (jb > 0 && ((keys[mid + jb - 1] & lowmask) >> w) == v) --jb;
    }
    d.ia = s + i; d.ib = mid + jb;
    desc[j] = d;
}

// ---------------------------------------------------------------------------------------
// shared pieces of the tile kernels
// ---------------------------------------------------------------------------------------
struct Pieces { u64 s0, s1, s2; u32 l0, l1, l2; };

__device__ __forceinline__ Pieces tile_pieces(const TileDesc& d0, const TileDesc& d1) {
    Pieces pc;
    if (d0.e == d1.e) {   // both boundaries in one block
        pc.s0 = d0.ia; pc.l0 = (u32)(d1.ia - d0.ia);
        pc.s1 = d0.ib; pc.l1 = (u32)(d1.ib - d0.ib);
        pc.s2 = 0; pc.l2 = 0;
    } else {              // A tail | B tail + whole blocks + A head | B head
        pc.s0 = d0.ia; pc.l0 = (u32)(d0.mid - d0.ia);
        pc.s1 = d0.ib; pc.l1 = (u32)(d1.ia - d0.ib);
        pc.s2 = d1.mid; pc.l2 = (u32)(d1.ib - d1.mid);
    }
    return pc;
}

__device__ __forceinline__ u64 piece_index(const Pieces& pc, u32 idx) {
    if (idx < pc.l0) return pc.s0 + idx;
    idx -= pc.l0;
    if (idx < pc.l1) return pc.s1 + idx;
    return pc.s2 + (idx - pc.l1);
}

__device__ __forceinline__ u64 moved_key(u64 k, int p, u64 himask, u64 lowmask) {
    return (k & himask) | ((k & lowmask) << 1) | ((k >> p) & 1ull);
}

// In-tile segmented merge.  sk[0..cnt) holds the tile's keys ascending in the OLD order.
// Each thread owns VT consecutive elements, finds the partner run of its run by binary
// search once and then advances a cursor.  emit(i, rank) is called with the element's
// rank in the NEW order (bit p moved to the LSB).  aux: run starts (cnt+2 entries).
template <int VT, typename Emit>
__device__ __forceinline__ void tile_merge(const u64* sk, unsigned short* aux, int* red, int cnt, int p, Emit emit) {
    const int tid = threadIdx.x;
    const int i0 = min(cnt, tid * VT), i1 = min(cnt, i0 + VT);
    const u64 lowmask = (1ull << p) - 1;
    int nh = 0;
    for (int i = i0; i < i1; ++i) nh += (i == 0) || ((sk[i] >> p) != (sk[i - 1] >> p));
    int nruns;
    const int excl = block_excl_scan(nh, red, &nruns);
    {
        int r = excl;
        for (int i = i0; i < i1; ++i)
            if ((i == 0) || ((sk[i] >> p) != (sk[i - 1] >> p))) aux[r++] = (unsigned short)i;
        if (tid == 0) { aux[nruns] = (unsigned short)cnt; aux[nruns + 1] = (unsigned short)cnt; }
    }
    __syncthreads();
    int run = excl - 1;
    int q = 0, plo = 0, phi = 0;
    bool fresh = true;
    for (int i = i0; i < i1; ++i) {
        const u64 k = sk[i];
        const bool head = (i == 0) || ((k >> p) != (sk[i - 1] >> p));
        if (head) { ++run; fresh = true; }
        const u64 low = k & lowmask;
        const int b = (int)((k >> p) & 1ull);
        if (fresh) {
            fresh = false;
            const int rs = aux[run], re = aux[run + 1];
            const u64 pre = (p == 63) ? 0 : (k >> (p + 1));
            if (b == 0) {
                plo = re; phi = re;
                if (re < cnt) {
                    const u64 pk = sk[re];
                    if (((p == 63) ? 0 : (pk >> (p + 1))) == pre) phi = aux[run + 2];
                }
                int lo = plo, hi = phi;   // first partner element with low >= mine
                while (lo < hi) { int m = (lo + hi) >> 1; if ((sk[m] & lowmask) < low) lo = m + 1; else hi = m; }
                q = lo;
            } else {
                plo = rs; phi = rs;
                if (rs > 0) {
                    const u64 pk = sk[rs - 1];
                    if (((p == 63) ? 0 : (pk >> (p + 1))) == pre) plo = aux[run - 1];
                }
                int lo = plo, hi = phi;   // first partner element with low > mine
                while (lo < hi) { int m = (lo + hi) >> 1; if ((sk[m] & lowmask) <= low) lo = m + 1; else hi = m; }
                q = lo;
            }
        } else if (b == 0) {
            while (q < phi && (sk[q] & lowmask) < low) ++q;
        } else {
            while (q < phi && (sk[q] & lowmask) <= low) ++q;
        }
        const int rank = (b == 0) ? i + (q - plo) : i - (phi - q);
        emit(i, rank);
    }
}

// ---------------------------------------------------------------------------------------
// pure bit move: same terms, new physical order (state preserving)
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SV_THREADS) move_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                          u64* __restrict__ kout, double2* __restrict__ aout,
                                                          int p, const TileDesc* __restrict__ desc) {
    constexpr int TCAP = SV_MOVE_TILE;
    constexpr int VT = TCAP / SV_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* sa = reinterpret_cast<double2*>(smem_raw);
    u64* sk = reinterpret_cast<u64*>(sa + TCAP);
    unsigned short* src = reinterpret_cast<unsigned short*>(sk + TCAP);
    unsigned short* aux = src + TCAP;
    __shared__ int red[SV_THREADS / 32 + 2];
    const int tid = threadIdx.x;
    const TileDesc d0 = desc[blockIdx.x], d1 = desc[blockIdx.x + 1];
    const Pieces pc = tile_pieces(d0, d1);
    const int cnt = min((u32)TCAP, pc.l0 + pc.l1 + pc.l2);
    for (int idx = tid; idx < cnt; idx += SV_THREADS) {
        const u64 g = piece_index(pc, idx);
        sk[idx] = ld_stream_u64(kin + g);
        sa[idx] = ld_stream_d2(ain + g);
    }
    __syncthreads();
    tile_merge<VT>(sk, aux, red, cnt, p, [&](int i, int rank) { src[rank] = (unsigned short)i; });
    __syncthreads();
    const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = (1ull << p) - 1;
    const u64 base = d0.ia + d0.ib - d0.mid;   // rank of the tile's first output
    for (int r = tid; r < cnt; r += SV_THREADS) {
        const int i = src[r];
        st_stream_u64(kout + base + r, moved_key(sk[i], p, himask, lowmask));
        st_stream_d2(aout + base + r, sa[i]);
    }
}

int svk_find_splits(const u64* keys, u64 n, int p, int w, u32 tnom, u32 ntiles, TileDesc* desc, cudaStream_t st) {
    const u32 nb = (ntiles + 1 + 127) / 128;
    find_splits_kernel<<<nb, 128, 0, st>>>(keys, n, p, w, tnom, ntiles, desc);
    return 1;
}

int svk_move(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, TileDesc* desc,
             cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1) {
    if (n == 0) return 0;
    const u32 ntiles = (u32)((n + SV_MOVE_TILE - 1) / SV_MOVE_TILE);
    int l = svk_find_splits(kin, n, p, -1, SV_MOVE_TILE, ntiles, desc, st);
    const size_t smem = (size_t)SV_MOVE_TILE * (16 + 8 + 2) + (SV_MOVE_TILE + 2) * 2;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(move_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr = true; }
    if (e0) cudaEventRecord(e0, st);
    move_kernel<<<ntiles, SV_THREADS, smem, st>>>(kin, ain, kout, aout, p, desc);
    if (e1) cudaEventRecord(e1, st);
    return l + 1;
}

// ---------------------------------------------------------------------------------------
// final pass of a group gate: (optional last move) + tuple formation + mat-vec + zero
// drop + stable compaction (decoupled look-back)
// ---------------------------------------------------------------------------------------
template <int MA, bool MOVE>
__global__ void __launch_bounds__(SV_THREADS) group_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                           u64* __restrict__ kout, double2* __restrict__ aout, u64 n,
                                                           int p, const GateTab* __restrict__ gtab,
                                                           const TileDesc* __restrict__ desc, u64* status,
                                                           u32* tile_counter, u64* d_count, u64 cap, u32 ntiles) {
    constexpr int TCAP = SV_TILE_SLOTS >> MA;
    constexpr int TNOM = TCAP - (1 << MA);
    constexpr int VT = (TCAP + SV_THREADS - 1) / SV_THREADS;
    constexpr int NIT = SV_TILE_SLOTS / SV_THREADS;
    constexpr u64 AM = (1ull << MA) - 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* sa = reinterpret_cast<double2*>(smem_raw);
    u64* sk2 = reinterpret_cast<u64*>(sa + TCAP);
    u64* sk = sk2 + TCAP;                                   // MOVE only
    unsigned short* src = reinterpret_cast<unsigned short*>(sk + (MOVE ? TCAP : 0));   // MOVE only
    unsigned short* aux = src + (MOVE ? TCAP : 0);          // TCAP + 2
    __shared__ int red[SV_THREADS / 32 + 2];
    __shared__ int wcnt[NIT][SV_THREADS / 32];
    __shared__ u32 s_tile;
    __shared__ u64 s_base;
    __shared__ u64 s_rng[2];
    __shared__ double2 sU[256];
    __shared__ int s_cpos[SV_MAX_M], s_col[16], s_mc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) s_tile = atomicAdd(tile_counter, 1u);
    for (int i = tid; i < 256; i += SV_THREADS) sU[i] = gtab->U[i];
    if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
    if (tid < 16) s_col[tid] = gtab->colorder[tid];
    if (tid == 0) s_mc = gtab->mc;
    __syncthreads();
    const u32 tile = s_tile;
    int cnt;
    if (MOVE) {
        const TileDesc d0 = desc[tile], d1 = desc[tile + 1];
        const Pieces pc = tile_pieces(d0, d1);
        cnt = min((u32)TCAP, pc.l0 + pc.l1 + pc.l2);
        for (int idx = tid; idx < cnt; idx += SV_THREADS) {
            const u64 g = piece_index(pc, idx);
            sk[idx] = ld_stream_u64(kin + g);
            sa[idx] = ld_stream_d2(ain + g);
        }
        __syncthreads();
        const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = (1ull << p) - 1;
        tile_merge<VT>(sk, aux, red, cnt, p, [&](int i, int rank) {
            src[rank] = (unsigned short)i;
            sk2[rank] = moved_key(sk[i], p, himask, lowmask);
        });
        __syncthreads();
    } else {
        if (tid < 2) {   // contiguous tile, boundaries pulled back to a tuple start
            u64 t = (u64)(tile + tid) * TNOM;
            if (t >= n) t = n;
            else if (t > 0) {
                const u64 v = kin[t] >> MA;
                while (t > 0 && (kin[t - 1] >> MA) == v) --t;
            }
            s_rng[tid] = t;
        }
        __syncthreads();
        const u64 a0 = s_rng[0];
        cnt = (int)min((u64)TCAP, s_rng[1] - a0);
        for (int idx = tid; idx < cnt; idx += SV_THREADS) {
            sk2[idx] = ld_stream_u64(kin + a0 + idx);
            sa[idx] = ld_stream_d2(ain + a0 + idx);
        }
        __syncthreads();
    }

    // tuple heads -> aux[g] = first element of tuple g
    const int i0 = min(cnt, tid * VT), i1 = min(cnt, i0 + VT);
    int nh = 0;
    for (int i = i0; i < i1; ++i) nh += (i == 0) || ((sk2[i] >> MA) != (sk2[i - 1] >> MA));
    int ngroups;
    const int gex = block_excl_scan(nh, red, &ngroups);   // (its barriers also retire the merge's use of aux)
    {
        int g = gex;
        for (int i = i0; i < i1; ++i)
            if ((i == 0) || ((sk2[i] >> MA) != (sk2[i - 1] >> MA))) aux[g++] = (unsigned short)i;
        if (tid == 0) aux[ngroups] = (unsigned short)cnt;
    }
    __syncthreads();

    // one thread per output slot (tuple g, row xr): out = sum_c U[xr][c] a[c], c ascending logical
    const int nslots = ngroups << MA;
    const int mc = s_mc;
    double outr[NIT], outi[NIT];
    u32 ball[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int slot = it * SV_THREADS + tid;
        double sr = 0.0, si = 0.0;
        bool flag = false;
        if (slot < nslots) {
            const int g = slot >> MA, xr = slot & (int)AM;
            const int gs = aux[g], ge = aux[g + 1];
            const u64 bk = sk2[gs];
            int cx = 0;
            for (int j = 0; j < mc; ++j) cx |= (int)((bk >> s_cpos[j]) & 1ull) << j;
            u32 pm = 0;
            for (int r = gs; r < ge; ++r) pm |= 1u << (u32)(sk2[r] & AM);
            const double2* urow = &sU[((cx << MA) | xr) << MA];
#pragma unroll
            for (int t = 0; t < (1 << MA); ++t) {
                const int x = (MA == 0) ? 0 : s_col[t];
                if ((pm >> x) & 1u) {
                    const int r = gs + __popc(pm & ((1u << x) - 1u));
                    const double2 a = sa[MOVE ? (int)src[r] : r];
                    const double2 u = urow[x];
                    cmul_acc(sr, si, u.x, u.y, a.x, a.y);
                }
            }
            flag = !(sr == 0.0 && si == 0.0);   // only nonzero amplitudes are stored
        }
        outr[it] = sr; outi[it] = si;
        const u32 b = __ballot_sync(0xffffffffu, flag);
        ball[it] = b;
        if (lane == 0) wcnt[it][warp] = __popc(b);
    }
    __syncthreads();
    if (tid == 0) {   // exclusive offsets of the NIT x 8 warp counts, tile total, look-back
        int run = 0;
        for (int it = 0; it < NIT; ++it)
            for (int w = 0; w < SV_THREADS / 32; ++w) { const int c = wcnt[it][w]; wcnt[it][w] = run; run += c; }
        const u64 excl = lookback_exclusive(status, tile, (u64)run);
        s_base = excl;
        if (tile == ntiles - 1) *d_count = excl + (u64)run;
    }
    __syncthreads();
    const u64 base = s_base;
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int slot = it * SV_THREADS + tid;
        if ((ball[it] >> lane) & 1u) {
            const u64 pos = base + (u64)wcnt[it][warp] + (u64)__popc(ball[it] & ((1u << lane) - 1u));
            if (pos < cap) {
                const u64 bk = sk2[aux[slot >> MA]];
                st_stream_u64(kout + pos, (bk & ~AM) | (u64)(slot & (int)AM));
                double2 o; o.x = outr[it]; o.y = outi[it];
                st_stream_d2(aout + pos, o);
            }
        }
    }
}

template <int MA, bool MOVE>
static void launch_group(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p,
                         const GateTab* tab, TileDesc* desc, u64* status, u32* tile_counter, u64* d_count, u64 cap,
                         u32 ntiles, cudaStream_t st) {
    constexpr int TCAP = SV_TILE_SLOTS >> MA;
    const size_t smem = (size_t)TCAP * (16 + 8) + (MOVE ? (size_t)TCAP * (8 + 2) : 0) + (TCAP + 2) * 2 + 16;
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(group_kernel<MA, MOVE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr = true;
    }
    group_kernel<MA, MOVE><<<ntiles, SV_THREADS, smem, st>>>(kin, ain, kout, aout, n, p, tab, desc, status,
                                                            tile_counter, d_count, cap, ntiles);
}

int svk_group(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int ma,
              const GateTab* tab, TileDesc* desc, u64* status, u32* tile_counter, u64* d_count, u64 cap,
              cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1) {
    int launches = 0;
    if (n == 0) { cudaMemsetAsync(d_count, 0, sizeof(u64), st); return 0; }
    const u32 tnom = (u32)((SV_TILE_SLOTS >> ma) - (1 << ma));
    const u32 ntiles = (u32)((n + tnom - 1) / tnom);
    cudaMemsetAsync(status, 0, (size_t)ntiles * sizeof(u64), st);
    cudaMemsetAsync(tile_counter, 0, sizeof(u32), st);
    const bool mv = p >= 0;
    if (mv) launches += svk_find_splits(kin, n, p, ma - 1, tnom, ntiles, desc, st);
    if (e0) cudaEventRecord(e0, st);
#define SV_LG(MA_) \
    if (mv) launch_group<MA_, true>(kin, ain, kout, aout, n, p, tab, desc, status, tile_counter, d_count, cap, ntiles, st); \
    else launch_group<MA_, false>(kin, ain, kout, aout, n, p, tab, desc, status, tile_counter, d_count, cap, ntiles, st);
    switch (ma) {
        case 0: SV_LG(0) break;
        case 1: SV_LG(1) break;
        case 2: SV_LG(2) break;
        case 3: SV_LG(3) break;
        default: SV_LG(4) break;
    }
#undef SV_LG
    if (e1) cudaEventRecord(e1, st);
    return launches + 1;
}
