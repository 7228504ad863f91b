// join.cu — S3a/K3: run boundaries and candidate-pair emission, as a shared-memory hash join over
// the buckets left by the radix partition.
//
// "Use the sorted array to identify groups of input strings that generate identical deletion
// variants, and transform this to an array of neighbor candidates" (App. F.2 step 3);
// "For each group v_g, generate all possible matching sequence pairs {(i', i'')} within the group"
// (App. F.3 step 3); a variant shared by m sequences yields m(m-1)/2 pairs
// (PAPER.md:96).  Output slots are allocated by prefix sums before anything is written ("avoid race
// condition by preallocating the outputs", Fig. S8).
//
// The records arrive partitioned on their top `sort_bits` hash bits only (S2 stops there): a BUCKET is
// a maximal range of records agreeing on those bits, a few thousand records by construction.  Equal
// variants always share a bucket, so the join is local to it: a block loads whole buckets into shared
// memory and
//   1. filters: every record sets one bit of a "seen" bitmap addressed by the next 16 hash bits and,
//      if it was already set, the same bit of a "seen twice" bitmap; only records whose "seen twice"
//      bit is set can have a partner (a few per cent on sparse data) — one atomic per record;
//   2. compacts those records, in position order, into a list;
//   3. chains the listed records by further hash bits (one atomic exchange each) and lets each walk its
//      chain for EARLIER records with the same full hash.
// The remaining sort passes over all records and the read of the sorted array are replaced by one read.
// Neither the order of the records inside a bucket nor the order of the buckets matters.
//
// Work split: tile t owns the buckets that START in [t*T, (t+1)*T).  It loads T + slack records, finds
// the first bucket boundary at or after each end of its range and joins what lies between.  A region
// that does not fit (a huge bucket: one variant shared by many thousands of sequences) is processed in
// chunks: build the table on a chunk, join it with itself, then stream the rest of its last bucket
// through the table.
//
// Numbering: a record's pairs get consecutive flat indices (thread-local order is fixed by the record
// positions, so it is the same in every round); a round writes the records whose FIRST index lies in
// [win_lo, win_hi), whole, at cand[index - win_lo] — the buffer keeps n_total + 64 slots of slack for
// the overhang — and reports the end of what it wrote in info->win_end, where the next round starts.
#include <cstddef>
#include <type_traits>

#include "kernels.h"


namespace {

constexpr int JN_THREADS = 512, JN_NW = JN_THREADS / 32, JN_T = 4096, JN_CAP = 6144;
constexpr int JN_IT = JN_CAP / JN_THREADS;                     // strided iterations that cover a full window
constexpr int JN_SLOT_BITS = 12, JN_SLOTS = 1 << JN_SLOT_BITS;  // chain heads
constexpr int JBM_BITS = 16;  // filter bitmap: 2^JBM_BITS bits each ("seen", "seen twice"); 15 bits: +6 %, 14 bits: +16 % on config 3
constexpr int JN_BM_BITS = JBM_BITS, JN_BM_WORDS = (1 << JN_BM_BITS) / 32;
constexpr u32 JN_NIL = 0xffffu, JN_NONE = 0xffffffffu;
static_assert(JN_CAP < 0xffff && JN_CAP % JN_THREADS == 0 && JN_IT <= 32, "node index / nzmask width");

struct JoinParams {
    const u64* rec;
    u64 n;
    u64 topmask;  // the radix-partitioned bits: a bucket = maximal range agreeing on them (0: one bucket)
    u64 hlim;     // 1 << id_bits: same hash <=> (x ^ y) < hlim
    u64 idmask, n_a;
    int bm_shift, slot_shift, b_bits, cross;
    u64* cand;
    u64 cand_cap;  // physical slots of cand
    u64 win_lo, win_hi;
    int first_round;
    u64* tile_prefix;
    DevInfo* info;
};

__device__ __forceinline__ bool jn_pair(u64 x, u64 y, const JoinParams& P, u64& packed) {
    const u64 a = x & P.idmask, b = y & P.idmask;
    if (P.cross) {
        const bool ax = a < P.n_a, bx = b < P.n_a;
        if (ax == bx) return false;
        packed = ((ax ? a : b) << P.b_bits) | ((ax ? b : a) - P.n_a);
    } else {
        if (a == b) return false;  // one sequence twice under one key (thinning off, or a hash collision)
        packed = (min(a, b) << P.b_bits) | max(a, b);
    }
    return true;
}

struct JoinSmem {
    u64 rec[JN_CAP + 2];     // [0] = record before the window, [1 + r] = record sb + r
    u32 bit_a[JN_BM_WORDS];  // seen
    u32 bit_b[JN_BM_WORDS];  // seen twice
    u32 head[JN_SLOTS];      // chain heads (window position of the last listed record of the slot)
    unsigned short next[JN_CAP];
    unsigned short list[JN_CAP];  // window positions of the records that may have a partner, ascending
    u64 wsum[JN_NW];
    u64 excl;
    u32 wcnt[JN_NW];
    u32 lo, hi;
};

__global__ void __launch_bounds__(JN_THREADS, 2) k_join(const JoinParams P) {
    extern __shared__ __align__(16) unsigned char jn_smem[];
    JoinSmem& S = *reinterpret_cast<JoinSmem*>(jn_smem);

    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 lane_lt = (1u << lane) - 1u;
    const u32 tile = blockIdx.x;
    if (!P.first_round) {
        const u64 lo = P.tile_prefix[2 * tile], cnt = P.tile_prefix[2 * tile + 1];
        if (cnt == 0 || lo + cnt <= P.win_lo || lo >= P.win_hi) return;  // nothing of this tile starts in the window
    }
    const u64 N = P.n;
    const u64 g0 = (u64)tile * JN_T;
    const u64 E = min(g0 + (u64)JN_T, N);  // the region ends at the first boundary >= E

    // loads records [sb - 1, sb + CAP] (one before, one lookahead) and returns the usable count W
    auto load = [&](u64 sb) -> u32 {
        const u32 cnt = (u32)min((u64)(JN_CAP + 1), N - sb);
        for (u32 r = tid; r < cnt; r += JN_THREADS) S.rec[1 + r] = P.rec[sb + r];
        if (tid == 0) S.rec[0] = sb > 0 ? P.rec[sb - 1] : 0ull;
        return min(cnt, (u32)JN_CAP);
    };
    // position sb + r starts a bucket (r in [0, W]; position N counts as a boundary)
    auto isb = [&](u64 sb, u32 r) -> bool {
        const u64 g = sb + r;
        return g == 0 || g == N || ((S.rec[r] ^ S.rec[1 + r]) & P.topmask) != 0;
    };
    auto slot_of = [&](u64 x) -> u32 { return (u32)(x >> P.slot_shift) & (JN_SLOTS - 1); };

    // Lists the window positions in [r0, r1) that may have a partner (filter: only those whose "seen
    // twice" bit is set; else all), ascending, and chains the listed records.  Every warp owns a
    // contiguous span, so the list order is the position order whatever the timing.
    auto prepare = [&](u32 r0, u32 r1, bool filter) -> u32 {
        for (u32 i = tid; i < JN_SLOTS / 4; i += JN_THREADS)
            reinterpret_cast<uint4*>(S.head)[i] = make_uint4(JN_NIL, JN_NIL, JN_NIL, JN_NIL);
        if (filter)
            for (u32 i = tid; i < 2 * JN_BM_WORDS / 4; i += JN_THREADS)
                reinterpret_cast<uint4*>(S.bit_a)[i] = make_uint4(0u, 0u, 0u, 0u);  // bit_a and bit_b are adjacent
        __syncthreads();
        const u32 span = (r1 - r0 + JN_THREADS - 1) / JN_THREADS * 32;  // per warp, a multiple of 32, <= 32 * JN_IT
        const u32 wbeg = r0 + warp * span;
        u32 bal[JN_IT];
        u32 cnt = 0;
        if (filter) {
            u32 bm[JN_IT];
#pragma unroll
            for (int it = 0; it < JN_IT; ++it) {
                const u32 r = wbeg + it * 32 + lane;
                bm[it] = JN_NONE;
                if ((u32)(it * 32) < span && r < r1) {
                    const u32 b = (u32)(S.rec[1 + r] >> P.bm_shift) & ((1u << JN_BM_BITS) - 1u);
                    bm[it] = b;
                    const u32 bit = 1u << (b & 31u);
                    if (atomicOr(&S.bit_a[b >> 5], bit) & bit) atomicOr(&S.bit_b[b >> 5], bit);
                }
            }
            __syncthreads();
#pragma unroll
            for (int it = 0; it < JN_IT; ++it) {
                const bool c = bm[it] != JN_NONE && ((S.bit_b[bm[it] >> 5] >> (bm[it] & 31u)) & 1u);
                bal[it] = __ballot_sync(SD_FULL, c);
                cnt += __popc(bal[it]);
            }
        } else {
#pragma unroll
            for (int it = 0; it < JN_IT; ++it) {
                const bool c = (u32)(it * 32) < span && wbeg + it * 32 + lane < r1;
                bal[it] = __ballot_sync(SD_FULL, c);
                cnt += __popc(bal[it]);
            }
        }
        if (lane == 0) S.wcnt[warp] = cnt;
        __syncthreads();
        u32 base = 0, total = 0;
#pragma unroll
        for (int w = 0; w < JN_NW; ++w) {
            const u32 c = S.wcnt[w];
            if ((u32)w < warp) base += c;
            total += c;
        }
#pragma unroll
        for (int it = 0; it < JN_IT; ++it) {
            if ((bal[it] >> lane) & 1u) S.list[base + __popc(bal[it] & lane_lt)] = (unsigned short)(wbeg + it * 32 + lane);
            base += __popc(bal[it]);
        }
        __syncthreads();
        for (u32 i = tid; i < total; i += JN_THREADS) {
            const u32 r = S.list[i];
            S.next[r] = (unsigned short)atomicExch(&S.head[slot_of(S.rec[1 + r])], r);
        }
        __syncthreads();
        return total;
    };

    u64 wend = 0;
    // pairs of record x with the chained records at window positions < lim; returns their number and,
    // when `store`, writes them from cand[at]
    auto walk = [&](u64 x, u32 lim, bool store, u64 at) -> u32 {
        u32 c = 0;
        for (u32 j = S.head[slot_of(x)]; j != JN_NIL; j = S.next[j]) {
            if (j < lim) {
                const u64 y = S.rec[1 + j];
                u64 packed;
                if ((x ^ y) < P.hlim && jn_pair(x, y, P, packed)) {
                    if (store) {
                        if (at + c < P.cand_cap) P.cand[at + c] = packed;
                        else atomicOr(&P.info->err, (u32)SD_ERR_OVERFLOW);
                    }
                    ++c;
                }
            }
        }
        return c;
    };
    auto visit = [&](u64 x, u32 lim, bool write, u64& flat) -> u32 {
        const bool inwin = write && flat >= P.win_lo && flat < P.win_hi;
        const u32 c = walk(x, lim, inwin, flat - P.win_lo);
        flat += c;
        if (inwin && c) wend = max(wend, flat);
        return c;
    };

    // ---- first chunk: the window of this tile; which buckets start in it? ----
    if (tid == 0) S.lo = JN_NONE, S.hi = JN_NONE;
    u32 W = load(g0);
    __syncthreads();
    {
        u32 mlo = JN_NONE, mhi = JN_NONE;  // r ascends: keep the first of each kind
        for (u32 r = tid; r <= W; r += JN_THREADS)
            if (isb(g0, r)) {
                if (g0 + r < E) mlo = min(mlo, r);
                else mhi = min(mhi, r);
            }
        mlo = __reduce_min_sync(SD_FULL, mlo);
        mhi = __reduce_min_sync(SD_FULL, mhi);
        if (lane == 0 && mlo != JN_NONE) atomicMin(&S.lo, mlo);
        if (lane == 0 && mhi != JN_NONE) atomicMin(&S.hi, mhi);
    }
    __syncthreads();
    const u32 lo = S.lo, hi0 = S.hi;
    if (lo == JN_NONE) {  // no bucket starts here
        if (P.first_round && tid == 0) P.tile_prefix[2 * tile] = 0, P.tile_prefix[2 * tile + 1] = 0;
        return;
    }
    const bool single = hi0 != JN_NONE;  // the whole region sits in shared memory
    u32 nzmask = 0;                      // single: which of this thread's listed records have pairs

    u64 flat = 0;
    for (int phase = 0; phase < 2; ++phase) {
        const bool write = phase == 1;
        u64 sb = g0;
        u32 r0 = lo, r1 = single ? hi0 : (u32)JN_CAP;
        bool last = single;
        for (bool first = true;; first = false) {
            if (!first || (write && !single)) {  // an oversized region: (re)load the chunk that starts at sb
                __syncthreads();
                if (tid == 0) S.hi = JN_NONE;
                W = load(sb);
                __syncthreads();
                if (!first) {
                    u32 mhi = JN_NONE;
                    for (u32 r = 1 + tid; r <= W; r += JN_THREADS)
                        if (isb(sb, r)) mhi = min(mhi, r);
                    mhi = __reduce_min_sync(SD_FULL, mhi);
                    if (lane == 0 && mhi != JN_NONE) atomicMin(&S.hi, mhi);
                    __syncthreads();
                    last = S.hi != JN_NONE;
                    r0 = 0;
                    r1 = last ? S.hi : (u32)JN_CAP;
                }
            }
            // ---- the chunk with itself ----
            if (single && write) {
                for (u32 m = nzmask, k = 0; m; m >>= 1, ++k)
                    if (m & 1u) {
                        const u32 r = S.list[tid + k * JN_THREADS];
                        visit(S.rec[1 + r], r, true, flat);
                    }
            } else {
                // the filter needs whole buckets in the table: not when later records are streamed through it
                const u32 nl = prepare(r0, r1, single);
                u32 k = 0;
                for (u32 i = tid; i < nl; i += JN_THREADS, ++k) {
                    const u32 r = S.list[i];
                    if (visit(S.rec[1 + r], r, write, flat) && single) nzmask |= 1u << k;
                }
            }
            if (last) break;
            // ---- the rest of the chunk's last bucket against the chunk ----
            if (!isb(sb, JN_CAP)) {
                const u64 lastx = S.rec[JN_CAP];
                for (u64 q0 = sb + JN_CAP;; q0 += JN_THREADS) {
                    const u64 q = q0 + tid;
                    u64 x = 0;
                    bool inb = q < N;
                    if (inb) {
                        x = P.rec[q];
                        inb = ((x ^ lastx) & P.topmask) == 0;
                    }
                    if (inb) visit(x, JN_CAP, write, flat);
                    if (!__syncthreads_and(inb)) break;
                }
            }
            sb += JN_CAP;
        }
        if (write) break;

        // ---- block exclusive scan of the per-thread totals; the tile claims its index range ----
        const u64 tsum = flat;
        u64 inc = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 t = __shfl_up_sync(SD_FULL, inc, o);
            if (lane >= (u32)o) inc += t;
        }
        if (lane == 31) S.wsum[warp] = inc;
        __syncthreads();
        u64 carry = 0, T = 0;
#pragma unroll
        for (int w = 0; w < JN_NW; ++w) {
            const u64 c = S.wsum[w];
            if ((u32)w < warp) carry += c;
            T += c;
        }
        if (T == 0) {
            if (P.first_round && tid == 0) P.tile_prefix[2 * tile] = 0, P.tile_prefix[2 * tile + 1] = 0;
            return;
        }
        if (tid == 0) {
            u64 excl;
            if (P.first_round) {
                excl = (u64)atomicAdd((unsigned long long*)&P.info->n_cand, (unsigned long long)T);
                P.tile_prefix[2 * tile] = excl;
                P.tile_prefix[2 * tile + 1] = T;
            } else {
                excl = P.tile_prefix[2 * tile];
            }
            S.excl = excl;
        }
        __syncthreads();
        flat = S.excl + carry + inc - tsum;  // flat index of this thread's first pair
        if (single && (tsum == 0 || flat + tsum <= P.win_lo || flat >= P.win_hi)) break;  // nothing of mine in the window
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wend = max(wend, __shfl_xor_sync(SD_FULL, wend, o));
    if (lane == 0 && wend) atomicMax((unsigned long long*)&P.info->win_end, (unsigned long long)wend);
}


// =================================================================================================
// Fast path: k_join_fast.  Same join, for the common case — every pair of the call fits the candidate
// buffer (one window).  It keeps NO copy of the tile in shared memory: a tile streams its records
// twice (the second time from registers / L1 / L2),
//   1. "seen" / "seen twice" bitmaps as above (one shared-memory atomic per record),
//   2. the records whose "seen twice" bit is set (a few per cent on sparse data) are appended to a
//      shared-memory list,
//   3. the listed records are chained by further hash bits; each walks the part of its chain that was
//      inserted BEFORE it (an exchange-built chain is in reverse insertion order), so every unordered
//      pair is met exactly once,
//   4. count, block scan, ONE global atomic per tile claims the output range, second walk writes.
// No bucket boundary is searched: tile t owns the buckets that start in [t*T, (t+1)*T), i.e. the
// records of its range whose partitioned bits differ from those of record t*T - 1, plus the records
// after the range that continue its last bucket (streamed until the partitioned bits change).
// The order of the candidates is arbitrary (they are sorted next).
//
// Two instances: LMAX = 2048 listed records per tile (44 KB of shared memory: four tiles per SM) runs
// first; a tile whose list overflows (dense data: most records have partners) puts its number on a
// redo list, which the LMAX = 6144 instance then processes.  If a tile overflows even that, or the
// claims run past the window, info->join_fallback is raised and the host reruns the general kernel
// above, which windows the output and chunks oversized buckets.
//
// K32: the partitioned bits and the bitmap bits all sit in the high word of the record (the usual
// layout); the filter phases then work on 32-bit words and keep only those in registers.
constexpr int JF_THREADS = 512, JF_NW = JF_THREADS / 32;
constexpr int JF_BM_BITS = JBM_BITS, JF_BM_WORDS = (1 << JF_BM_BITS) / 32;

template <int LMAX, int SLOT_BITS>
struct JoinFastSmem {
    u64 list[LMAX];
    u32 bit_a[JF_BM_WORDS];
    u32 bit_b[JF_BM_WORDS];
    u32 head[1 << SLOT_BITS];
    unsigned short next[LMAX];
    u32 wsum[JF_NW];
    u32 nlist;
    u64 base;
};

struct JoinFastParams {
    JoinParams j;
    const u32* tiles;  // nullptr: tile = block index; else the redo list
    u32* redo;         // nullptr: a list overflow raises join_fallback; else tiles append themselves here
};

__device__ __forceinline__ u32 jf_atoms_add(u32* p, u32 v) {  // plain ATOMS.ADD (no compiler-inserted warp aggregation)
    u32 old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"((u32)__cvta_generic_to_shared(p)), "r"(v) : "memory");
    return old;
}

template <bool K32, int IT, int LMAX, int SLOT_BITS, int MINB>
__global__ void __launch_bounds__(JF_THREADS, MINB) k_join_fast(const JoinFastParams FP) {
    typedef typename std::conditional<K32, u32, u64>::type K;  // the part of a record the filter looks at
    typedef JoinFastSmem<LMAX, SLOT_BITS> Smem;
    constexpr int SLOTS = 1 << SLOT_BITS, LIT = (LMAX + JF_THREADS - 1) / JF_THREADS, T = JF_THREADS * IT;
    static_assert(LMAX < 0xffff && LIT <= 32 && IT % 2 == 0 && IT <= 32, "node index width / mask widths");
    extern __shared__ __align__(16) unsigned char jn_smem[];
    Smem& S = *reinterpret_cast<Smem*>(jn_smem);
    const JoinParams& P = FP.j;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 lane_lt = (1u << lane) - 1u;
    const u64 N = P.n;
    const u32 tile = FP.tiles ? FP.tiles[blockIdx.x] : blockIdx.x;
    const u64 g0 = (u64)tile * T;
    const u64 E = min(g0 + (u64)T, N);
    auto key_of = [&](u64 y) -> K { return K32 ? (K)(y >> 32) : (K)y; };
    const K topmask = key_of(P.topmask);
    const int bm_shift = K32 ? P.bm_shift - 32 : P.bm_shift;
    const K v0 = g0 > 0 ? (key_of(P.rec[g0 - 1]) & topmask) : (K)0;  // bucket of the record before the range
    const K v1 = key_of(P.rec[E - 1]) & topmask;                      // bucket that may continue after the range
    if (g0 > 0 && v1 == v0) return;                                   // no bucket starts here

    for (u32 i = tid; i < 2 * JF_BM_WORDS / 4; i += JF_THREADS)
        reinterpret_cast<uint4*>(S.bit_a)[i] = make_uint4(0u, 0u, 0u, 0u);  // bit_a and bit_b are adjacent
    for (u32 i = tid; i < SLOTS / 4; i += JF_THREADS)
        reinterpret_cast<uint4*>(S.head)[i] = make_uint4(JN_NIL, JN_NIL, JN_NIL, JN_NIL);
    if (tid == 0) S.nlist = 0;

    // ---- the range, two records per 16-byte load: item 2k + e of the thread is record 2*(tid + k*THREADS) + e ----
    const u64* const rp = P.rec + g0 + 2 * tid;
    K x[IT];
    u32 mine = 0;
    const bool full = E - g0 == (u64)T;
#pragma unroll
    for (int k = 0; k < IT / 2; ++k) {
        const u32 r = 2 * (tid + k * JF_THREADS);
        if (full || g0 + r + 1 < E) {
            const ulonglong2 t = *reinterpret_cast<const ulonglong2*>(rp + 2 * k * JF_THREADS);
            x[2 * k] = key_of(t.x), x[2 * k + 1] = key_of(t.y);
            mine |= 3u << (2 * k);
        } else if (g0 + r < E) {
            x[2 * k] = key_of(rp[2 * k * JF_THREADS]), x[2 * k + 1] = 0;
            mine |= 1u << (2 * k);
        } else {
            x[2 * k] = x[2 * k + 1] = 0;
        }
    }
    if (g0 > 0) {
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if ((x[k] & topmask) == v0) mine &= ~(1u << k);
    }
    __syncthreads();
    auto bm_of = [&](K y) -> u32 { return (u32)(y >> bm_shift) & ((1u << JF_BM_BITS) - 1u); };
    auto mark = [&](K y) {
        const u32 b = bm_of(y), bit = 1u << (b & 31u);
        if (atomicOr(&S.bit_a[b >> 5], bit) & bit) atomicOr(&S.bit_b[b >> 5], bit);
    };
    // ---- 1. bitmaps ----
#pragma unroll
    for (int k = 0; k < IT; ++k)
        if ((mine >> k) & 1u) mark(x[k]);
    // The records after the range that continue its last bucket: every warp walks its own strided
    // positions until none of its lanes is in the bucket any more (the records are sorted on these bits).
    for (u64 q = E + tid; __any_sync(SD_FULL, q < N); q += JF_THREADS) {
        bool in = false;
        if (q < N) {
            const K y = key_of(P.rec[q]);
            in = (y & topmask) == v1;
            if (in) mark(y);
        }
        if (!__any_sync(SD_FULL, in)) break;
    }
    __syncthreads();
    // ---- 2. list the records whose "seen twice" bit is set ----
    auto listed = [&](K y) -> bool {
        const u32 b = bm_of(y);
        return (S.bit_b[b >> 5] >> (b & 31u)) & 1u;
    };
    {
        u32 lm = 0;
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (((mine >> k) & 1u) && listed(x[k])) lm |= 1u << k;
        // lane l's listed records go to slots [sum of popc(lm) over lanes < l, ...)
        const u32 c = __popc(lm);
        u32 inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 t = __shfl_up_sync(SD_FULL, inc, o);
            if (lane >= (u32)o) inc += t;
        }
        u32 at = 0;
        if (lane == 31 && inc) at = jf_atoms_add(&S.nlist, inc);
        at = __shfl_sync(SD_FULL, at, 31) + inc - c;
        while (lm) {
            const int k = __ffs(lm) - 1;
            lm &= lm - 1;
            if (at < (u32)LMAX) S.list[at] = rp[(k >> 1) * (2 * JF_THREADS) + (k & 1)];
            ++at;
        }
    }
    for (u64 q = E + tid; __any_sync(SD_FULL, q < N); q += JF_THREADS) {
        bool in = false, c = false;
        u64 y = 0;
        if (q < N) {
            y = P.rec[q];
            in = (key_of(y) & topmask) == v1;
            c = in && listed(key_of(y));
        }
        if (!__any_sync(SD_FULL, in)) break;
        const u32 bal = __ballot_sync(SD_FULL, c);
        if (bal) {
            u32 at = 0;
            if (lane == 0) at = jf_atoms_add(&S.nlist, (u32)__popc(bal));
            at = __shfl_sync(SD_FULL, at, 0) + __popc(bal & lane_lt);
            if (c && at < (u32)LMAX) S.list[at] = y;
        }
    }
    __syncthreads();
    const u32 nl = S.nlist;
    if (nl == 0) return;
    if (nl > (u32)LMAX) {
        if (tid == 0) {
            if (FP.redo) FP.redo[atomicAdd(&P.info->join_redo, 1u)] = tile;
            else atomicOr(&P.info->join_fallback, 1u);
        }
        return;
    }
    // ---- 3. chains ----
    auto slot_of = [&](u64 y) -> u32 { return (u32)(y >> P.slot_shift) & (SLOTS - 1); };
    for (u32 i = tid; i < nl; i += JF_THREADS) S.next[i] = (unsigned short)atomicExch(&S.head[slot_of(S.list[i])], i);
    __syncthreads();
    // ---- 4. count, claim, write ----
    u32 cnt = 0, nzmask = 0;
    {
        u32 k = 0;
        for (u32 i = tid; i < nl; i += JF_THREADS, ++k) {
            u32 j = S.next[i];
            if (j == JN_NIL) continue;
            const u64 y = S.list[i];
            u32 c = 0;
            for (; j != JN_NIL; j = S.next[j]) {
                const u64 z = S.list[j];
                u64 packed;
                if ((y ^ z) < P.hlim && jn_pair(y, z, P, packed)) ++c;
            }
            if (c) nzmask |= 1u << k;
            cnt += c;
        }
    }
    if (!__syncthreads_or(cnt != 0)) return;
    u32 inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 t = __shfl_up_sync(SD_FULL, inc, o);
        if (lane >= (u32)o) inc += t;
    }
    if (lane == 31) S.wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const u32 w = lane < JF_NW ? S.wsum[lane] : 0u;
        u32 winc = w;
#pragma unroll
        for (int o = 1; o < JF_NW; o <<= 1) {
            const u32 t = __shfl_up_sync(SD_FULL, winc, o);
            if (lane >= (u32)o) winc += t;
        }
        if (lane < JF_NW) S.wsum[lane] = winc - w;
        if (lane == JF_NW - 1) {
            const u64 base = (u64)atomicAdd((unsigned long long*)&P.info->n_cand, (unsigned long long)winc);
            // does not fit the window: nothing is written
            if (base + winc > P.win_hi) atomicOr(&P.info->join_fallback, 2u), S.base = ~0ull;
            else S.base = base;
        }
    }
    __syncthreads();
    if (S.base == ~0ull) return;
    u64 at = S.base + S.wsum[warp] + inc - cnt;
    for (u32 m = nzmask, k = 0; m; m >>= 1, ++k)
        if (m & 1u) {
            const u32 i = tid + k * JF_THREADS;
            const u64 y = S.list[i];
            for (u32 j = S.next[i]; j != JN_NIL; j = S.next[j]) {
                const u64 z = S.list[j];
                u64 packed;
                if ((y ^ z) < P.hlim && jn_pair(y, z, P, packed)) P.cand[at++] = packed;
            }
        }
}

constexpr int JF_IT = 8;      // records per thread of a k_join_fast tile
constexpr int JF_MINB_S = 4;  // resident blocks of the small-list instances
constexpr int JF_T = JF_THREADS * JF_IT;
constexpr int JF_LMAX_S = JF_IT > 8 ? 3072 : 2048, JF_SLOTB_S = 11;
constexpr int JF_LMAX_L = JF_T + 4096, JF_SLOTB_L = 12, JF_MINB_L = JF_IT > 8 ? 1 : 2;


// =================================================================================================
// Bucket join of the fused pipeline: k_join_bkt.  The level-2 partition leaves every bucket in its own
// fixed-capacity region with its record count, so nothing has to be found: ONE BLOCK PER BUCKET, and the
// bucket is joined in a single sweep by a chained hash table in shared memory:
//   0. the bucket comes into shared memory by one 1-D bulk asynchronous copy (cp.async.bulk, the TMA engine;
//      completion counted in bytes on an mbarrier) while the threads clear the chain heads — no per-thread
//      address arithmetic, no registers held across the phases;
//   1. sweep: every record swaps its position into the head of its slot (the hash bits right below the
//      partitioned ones; one shared-memory atomic exchange) and keeps the previous head as its `next` — IN the
//      staged record: its top NB bits are the same for the whole bucket (partitioned hash bits, or zeros above a
//      narrowed hash), so they carry the link and a chain step is ONE 8-byte shared load.  A record that found its
//      slot empty (about four in five on sparse data) is finished: whoever pairs with it comes LATER and will find it;
//   2. the others walk their chain — the records inserted BEFORE them — comparing the rest of the hash, so every
//      unordered pair is met exactly once, by its later member: count, ONE shared atomic per thread with pairs +
//      ONE global atomic per block claim the output range ("preallocating the outputs"), second
//      walk writes.
// No bitmaps, no candidate list, no list overflow: dense buckets (every record with partners) take the same
// path, their chains are just longer.  The kernel is latency-bound (dependent shared-memory accesses): what
// counts is resident warps, hence as little shared memory per block as the region needs: 16 KB of heads + the
// stage, sized at launch (config 3: 34 KB, six blocks of 256 threads per SM; with five blocks +12 %, with four
// +35 %).  Two instances: regions of up to 4064 records (NB = 12) and up to 18432 (1024 threads, NB = 15: chunks
// of more than ~2 * 10^8 records).
// Cross-search instance (CROSS): only the QUERY records are chained by atomic exchange (sweep 1a); every reference
// record then reads the head of its slot with a plain load and keeps it as its link (sweep 1b), so the walks run from
// reference records through query records only.
// Windowed searches (the pairs of a chunk exceed one candidate window).  A block claims its output range with ONE
// atomicAdd on info->n_cand, so the claims are totally ordered.  A claim that ends beyond the window (win_hi) writes
// nothing, marks its bucket open (JB_OPEN, bit 31 of the bucket's count), raises info->join_fallback and publishes its
// base through info->nofit_inv = max(~base): every claim after the first that does not fit starts beyond the window
// too, hence the pairs written are exactly [0, min base that did not fit) — the host takes that as the window's end
// and launches further passes (first_round = 0) that join only the open buckets, each into a fresh window; a bucket
// that fits clears its mark.  A bucket fuller than the launched instance stages (stage_cap) is left open the same way
// for a pass of the large instance.  Only a single bucket whose pairs exceed a whole window (a pass that writes
// nothing while buckets stay open) sends the chunk to the exact pipeline.
constexpr u32 JB_OPEN = 0x80000000u;
struct JoinBktParams {
    JoinParams j;       // rec = bucket regions; topmask unused
    u32* cnt;           // records per bucket; bit 31 = its pairs did not fit the window of an earlier pass (windowed searches: later passes join exactly these)
    u32 cap;            // region stride (records; a multiple of 32)
    u32 stage_cap;      // records the launched instance stages (<= cap): a fuller bucket is left open for a pass of the large instance
    u32 nbuckets;
};

// ---- bulk asynchronous copy + mbarrier (PTX; SASS: UBLKCP / SYNCS) ----
__device__ __forceinline__ u32 jb_smem(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void jb_mbar_init(u64* bar, u32 count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(jb_smem(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void jb_fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void jb_mbar_expect_tx(u64* bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(jb_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void jb_bulk_g2s(void* dst, const void* src, u32 bytes, u64* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(jb_smem(dst)),
                 "l"(src), "r"(bytes), "r"(jb_smem(bar))
                 : "memory");
}
__device__ __forceinline__ void jb_mbar_wait(u64* bar, u32 parity) {
    u32 done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(jb_smem(bar)), "r"(parity)
            : "memory");
    }
}
// (the address is a shared-window offset computed once per block: a generic pointer would cost a cvta per exchange)
__device__ __forceinline__ u32 jb_atoms_exch(u32 saddr, u32 v) {
    u32 old;
    asm volatile("atom.shared.exch.b32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v) : "memory");
    return old;
}

// shared memory: this header, then the stage (`cap` records, sized at launch: the smaller the regions, the more blocks per SM)
template <int SLOT_BITS>
struct JoinBktSmem {
    u32 head[1 << SLOT_BITS];  // last record inserted into the slot (all ones in NB bits: none)
    u64 mbar;
    u64 base;
    u32 total, pad[3];
    u64 stage[2];              // the bucket; after the sweep the top NB bits of a record = the record inserted into its slot before it
};

// STAGE_MAX: the largest region this instance accepts
template <int THREADS, int STAGE_MAX, int SLOT_BITS, int NB, int MINB, bool CROSS>
__global__ void __launch_bounds__(THREADS, MINB) k_join_bkt(const JoinBktParams BP) {
    typedef JoinBktSmem<SLOT_BITS> Smem;
    constexpr int SLOTS = 1 << SLOT_BITS, IT = (STAGE_MAX / 2 + THREADS - 1) / THREADS;  // 16-byte loads per thread that cover the stage
    constexpr u32 NIL = (1u << NB) - 1u;
    constexpr u64 KEEP = ~0ull >> NB;  // the bits of a staged record that are still the record
    static_assert(STAGE_MAX <= (int)NIL && STAGE_MAX % 2 == 0 && 2 * IT <= 32 && SLOTS % (4 * THREADS) == 0 && NB <= 16 &&
                      offsetof(Smem, stage) % 16 == 0, "link / flag mask widths");
    extern __shared__ __align__(16) unsigned char jn_smem[];
    Smem& S = *reinterpret_cast<Smem*>(jn_smem);
    const JoinParams& P = BP.j;
    const u32 tid = threadIdx.x;
    sd_dep_wait();  // (launched as a dependent of the level-2 partition)
    const u32 bucket = blockIdx.x;
    const u32 cword = BP.cnt[bucket];
    if (!P.first_round && !(cword & JB_OPEN)) return;  // later pass of a windowed search: only the buckets left open (block-uniform)
    const u32 n = min(cword & ~JB_OPEN, BP.cap);
    if (n < 2) return;  // nothing to pair
    if (n > BP.stage_cap) {  // (block-uniform) the small instance was launched on regions that may hold more than it stages
        if (tid == 0) {
            atomicOr(&P.info->join_fallback, 2u);
            if (!(cword & JB_OPEN)) BP.cnt[bucket] = cword | JB_OPEN;
        }
        return;
    }
    // later pass of a windowed search and the window is already full: this bucket waits for the next pass (nothing loaded,
    // nothing counted).  One thread looks, the barrier makes the decision the block's.
    if (!P.first_round && __syncthreads_or(tid == 0 && sd_ld_relaxed(&P.info->n_cand) >= P.win_hi)) {
        if (tid == 0) atomicOr(&P.info->join_fallback, 2u);
        return;
    }
    if (tid == 0) {
        S.total = 0;
        jb_mbar_init(&S.mbar, 1);
        jb_fence_proxy_async();
        const u32 bytes = ((n + 1u) & ~1u) * 8u;  // whole 16-byte units (the region is a multiple of 256 bytes)
        jb_mbar_expect_tx(&S.mbar, bytes);
        jb_bulk_g2s(S.stage, P.rec + (u64)bucket * BP.cap, bytes, &S.mbar);
    }
#pragma unroll
    for (int k = 0; k < SLOTS / (4 * THREADS); ++k)
        reinterpret_cast<uint4*>(S.head)[tid + k * THREADS] = make_uint4(NIL, NIL, NIL, NIL);
    __syncthreads();  // heads cleared, barrier initialised
    jb_mbar_wait(&S.mbar, 0);
    // ---- 1. sweep ----
    const int slot_shift = P.slot_shift;
    // The link goes into the top NB bits of the record and the PAIR of records is written back by one 16-byte store
    // (4 wavefronts per warp; two 2-byte stores at a 16-byte lane stride were 4-way bank conflicts: 8 wavefronts).
    const u32 head_s = jb_smem(S.head);
    u32 flag = 0;  // bit 2k + e: my record 2 * (tid + k * THREADS) + e found an earlier record in its slot
    if (!CROSS) {
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            const u32 i = 2 * (tid + k * THREADS);
            if (i < n) {
                ulonglong2 t = *reinterpret_cast<const ulonglong2*>(S.stage + i);
                const u32 o0 = jb_atoms_exch(head_s + 4u * ((u32)(t.x >> slot_shift) & (SLOTS - 1)), i);
                t.x = (t.x & KEEP) | ((u64)o0 << (64 - NB));
                flag |= (o0 != NIL ? 1u : 0u) << (2 * k);
                if (i + 1 < n) {
                    const u32 o1 = jb_atoms_exch(head_s + 4u * ((u32)(t.y >> slot_shift) & (SLOTS - 1)), i + 1);
                    t.y = (t.y & KEEP) | ((u64)o1 << (64 - NB));
                    flag |= (o1 != NIL ? 2u : 0u) << (2 * k);
                }
                *reinterpret_cast<ulonglong2*>(S.stage + i) = t;
            }
        }
    } else {
        // Cross-search: only (query, reference) pairs count, and the queries are usually the small side (config 4: 2 % of
        // the records).  Sweep 1a chains the QUERY records only; sweep 1b lets every reference record look at the head of
        // its slot — a plain load, no atomic, and nearly always empty — and keeps it as its link: the walk below then
        // runs from reference records through query records only.
        const u64 idm = P.idmask, na = P.n_a;
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            const u32 i = 2 * (tid + k * THREADS);
            if (i < n) {
                ulonglong2 t = *reinterpret_cast<const ulonglong2*>(S.stage + i);
                const bool q0 = (t.x & idm) < na, q1 = i + 1 < n && (t.y & idm) < na;
                if (q0) {
                    const u32 o0 = jb_atoms_exch(head_s + 4u * ((u32)(t.x >> slot_shift) & (SLOTS - 1)), i);
                    t.x = (t.x & KEEP) | ((u64)o0 << (64 - NB));
                }
                if (q1) {
                    const u32 o1 = jb_atoms_exch(head_s + 4u * ((u32)(t.y >> slot_shift) & (SLOTS - 1)), i + 1);
                    t.y = (t.y & KEEP) | ((u64)o1 << (64 - NB));
                }
                if (q0 || q1) *reinterpret_cast<ulonglong2*>(S.stage + i) = t;  // (queries are the small side: most pairs hold none)
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            const u32 i = 2 * (tid + k * THREADS);
            if (i < n) {
                ulonglong2 t = *reinterpret_cast<const ulonglong2*>(S.stage + i);  // (a query record keeps the link sweep 1a gave it: only `idm` bits are looked at)
                if ((t.x & idm) >= na) {
                    const u32 o0 = S.head[(u32)(t.x >> slot_shift) & (SLOTS - 1)];
                    t.x = (t.x & KEEP) | ((u64)o0 << (64 - NB));
                    flag |= (o0 != NIL ? 1u : 0u) << (2 * k);
                }
                if (i + 1 < n && (t.y & idm) >= na) {
                    const u32 o1 = S.head[(u32)(t.y >> slot_shift) & (SLOTS - 1)];
                    t.y = (t.y & KEEP) | ((u64)o1 << (64 - NB));
                    flag |= (o1 != NIL ? 2u : 0u) << (2 * k);
                }
                *reinterpret_cast<ulonglong2*>(S.stage + i) = t;
            }
        }
    }
    __syncthreads();
    // ---- 2. count, claim, write ----
    auto pos_of = [&](u32 e) -> u32 { return 2 * (tid + (e >> 1) * THREADS) + (e & 1u); };
    u32 cnt = 0, nz = 0;
    for (u32 m = flag; m; m &= m - 1) {
        const u32 e = __ffs(m) - 1;
        const u64 y = S.stage[pos_of(e)];
        u32 c = 0;
        if (!CROSS) {
            // self-search: same hash and different ids <=> 0 < (y ^ z) & KEEP < 2^id_bits
            for (u32 j = (u32)(y >> (64 - NB)); j != NIL;) {
                const u64 z = S.stage[j];
                c += (((y ^ z) & KEEP) - 1ull) < (P.hlim - 1ull) ? 1u : 0u;
                j = (u32)(z >> (64 - NB));
            }
        } else {
            for (u32 j = (u32)(y >> (64 - NB)); j != NIL;) {
                const u64 z = S.stage[j];
                u64 packed;
                if (((y ^ z) & KEEP) < P.hlim && jn_pair(y, z, P, packed)) ++c;
                j = (u32)(z >> (64 - NB));
            }
        }
        if (c) nz |= 1u << e;
        cnt += c;
    }
    u32 mine = 0;  // this thread's offset inside the block's output range (any order: the candidates are sorted next)
    if (cnt) mine = jf_atoms_add(&S.total, cnt);
    __syncthreads();
    const u32 total = S.total;
    if (total == 0) {
        if (tid == 0 && (cword & JB_OPEN)) BP.cnt[bucket] = cword & ~JB_OPEN;
        return;
    }
    if (tid == 0) {
        const u64 base = (u64)atomicAdd((unsigned long long*)&P.info->n_cand, (unsigned long long)total);
        // Does not fit the window: nothing is written, the bucket stays open for the next pass.  Claims are totally
        // ordered by the atomic: every claim after the first that does not fit starts beyond the window too, so the
        // pairs written are exactly [0, win_end) with win_end = the smallest base that did not fit.
        if (base + total > P.win_hi) {
            atomicOr(&P.info->join_fallback, 2u);
            atomicMax((unsigned long long*)&P.info->nofit_inv, (unsigned long long)~base);
            if (!(cword & JB_OPEN)) BP.cnt[bucket] = cword | JB_OPEN;
            S.base = ~0ull;
        } else {
            S.base = base;
            if (cword & JB_OPEN) BP.cnt[bucket] = cword & ~JB_OPEN;
        }
    }
    __syncthreads();
    if (S.base == ~0ull) return;
    u64 at = S.base + mine;
    for (u32 m = nz; m; m &= m - 1) {
        const u64 y = S.stage[pos_of(__ffs(m) - 1)];
        for (u32 j = (u32)(y >> (64 - NB)); j != NIL;) {
            const u64 z = S.stage[j];
            u64 packed;
            if (((y ^ z) & KEEP) < P.hlim && jn_pair(y, z, P, packed)) P.cand[at++] = packed;
            j = (u32)(z >> (64 - NB));
        }
    }
}

// the two instances: (threads, largest region, chain-head bits, link bits, resident blocks the registers must allow)
constexpr int JB_THREADS_S = 256, JB_STAGE_S = 4064, JB_SLOTB_S = 12, JB_NB_S = 12, JB_MINB_S = 6;
constexpr int JB_THREADS_L = 1024, JB_STAGE_L = 18432, JB_SLOTB_L = 13, JB_NB_L = 15, JB_MINB_L = 1;
static size_t jb_smem_bytes(bool small, u32 cap) {
    return (small ? offsetof(JoinBktSmem<JB_SLOTB_S>, stage) : offsetof(JoinBktSmem<JB_SLOTB_L>, stage)) + (size_t)cap * 8;
}
static_assert(6 * (offsetof(JoinBktSmem<JB_SLOTB_S>, stage) + 2304 * 8 + 1024) <= 233472, "six blocks per SM at config-3 regions (2304 records)");

}  // namespace

i64 sd_join_tiles(i64 n_records) { return (n_records + JN_T - 1) / JN_T; }

// Per-device state of this translation unit (dynamic shared-memory limits of the join kernels): set for the current
// device by every symdel_create — function attributes belong to a device, not to the process.
template <bool K32>
static cudaError_t jn_setup_k() {
    cudaError_t e;
    const int ss = (int)sizeof(JoinFastSmem<JF_LMAX_S, JF_SLOTB_S>), sl = (int)sizeof(JoinFastSmem<JF_LMAX_L, JF_SLOTB_L>);
    if ((e = cudaFuncSetAttribute(k_join_fast<K32, JF_IT, JF_LMAX_S, JF_SLOTB_S, JF_MINB_S>, cudaFuncAttributeMaxDynamicSharedMemorySize, ss)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_join_fast<K32, JF_IT, JF_LMAX_L, JF_SLOTB_L, JF_MINB_L>, cudaFuncAttributeMaxDynamicSharedMemorySize, sl)) != cudaSuccess) return e;
    return cudaSuccess;
}
cudaError_t sd_join_setup() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_join, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(JoinSmem))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_join_bkt<JB_THREADS_S, JB_STAGE_S, JB_SLOTB_S, JB_NB_S, JB_MINB_S, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)jb_smem_bytes(true, JB_STAGE_S))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_join_bkt<JB_THREADS_S, JB_STAGE_S, JB_SLOTB_S, JB_NB_S, JB_MINB_S, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)jb_smem_bytes(true, JB_STAGE_S))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_join_bkt<JB_THREADS_L, JB_STAGE_L, JB_SLOTB_L, JB_NB_L, JB_MINB_L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)jb_smem_bytes(false, JB_STAGE_L))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_join_bkt<JB_THREADS_L, JB_STAGE_L, JB_SLOTB_L, JB_NB_L, JB_MINB_L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)jb_smem_bytes(false, JB_STAGE_L))) != cudaSuccess) return e;
    if ((e = jn_setup_k<true>()) != cudaSuccess) return e;
    return jn_setup_k<false>();
}

static JoinParams jn_params(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 cand_cap, DevInfo* info) {
    JoinParams P{};
    P.rec = records;
    P.n = (u64)n_records;
    const int top = lay.id_bits + lay.hash_bits, sort_bits = lay.sort_bits;  // the hash field is bits [id_bits, top)
    P.topmask = sort_bits > 0 ? (~0ull >> (64 - sort_bits)) << (top - sort_bits) : 0ull;
    P.hlim = 1ull << lay.id_bits;
    P.idmask = P.hlim - 1ull;
    P.n_a = (u64)lay.n_a;
    // bitmap position = the hash bits right below the partitioned ones, chain slot = the bits below those
    // (both clamped to the hash field: with few hash bits they overlap, which only lengthens chains)
    P.bm_shift = std::max(lay.id_bits, top - sort_bits - JN_BM_BITS);
    P.slot_shift = std::max(lay.id_bits, P.bm_shift - JN_SLOT_BITS);
    P.b_bits = lay.b_bits;
    P.cross = lay.cross;
    P.cand = cand;
    P.cand_cap = cand_cap;
    P.info = info;
    return P;
}

// Fast path: all pairs in one window of `window` slots, arbitrary order; info->n_cand = total.
// Step 1 (sd_join_fast): the small-list instance over every tile; tiles whose list overflowed are in
// redo[0 .. info->join_redo).  Step 2 (sd_join_fast_redo, only if join_redo != 0): the large-list
// instance over those.  info->join_fallback != 0 after either: the general kernel has to redo the
// join (nothing usable was written).
template <bool K32>
static cudaError_t jn_launch_fast(const JoinFastParams& FP, unsigned grid, bool large, cudaStream_t st) {
    auto ks = k_join_fast<K32, JF_IT, JF_LMAX_S, JF_SLOTB_S, JF_MINB_S>;
    auto kl = k_join_fast<K32, JF_IT, JF_LMAX_L, JF_SLOTB_L, JF_MINB_L>;
    constexpr size_t ss = sizeof(JoinFastSmem<JF_LMAX_S, JF_SLOTB_S>), sl = sizeof(JoinFastSmem<JF_LMAX_L, JF_SLOTB_L>);
    if (large) kl<<<grid, JF_THREADS, sl, st>>>(FP);
    else ks<<<grid, JF_THREADS, ss, st>>>(FP);
    return cudaGetLastError();
}

static inline int jn_k32(const JoinParams& P) { return P.bm_shift >= 32 && (P.topmask & 0xffffffffull) == 0; }

cudaError_t sd_join_fast(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 window, u32* redo,
                         DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = (n_records + JF_T - 1) / JF_T;
    if (tiles == 0) return cudaSuccess;
    cudaError_t e;
    if ((e = cudaMemsetAsync(&info->n_cand, 0, sizeof(u64), st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&info->join_fallback, 0, 2 * sizeof(u32), st)) != cudaSuccess) return e;  // and join_redo
    JoinFastParams FP{};
    FP.j = jn_params(records, n_records, lay, cand, window, info);
    FP.j.win_lo = 0;
    FP.j.win_hi = window;
    FP.tiles = nullptr;
    FP.redo = redo;
    if (launches) ++*launches;
    return jn_k32(FP.j) ? jn_launch_fast<true>(FP, (unsigned)tiles, false, st) : jn_launch_fast<false>(FP, (unsigned)tiles, false, st);
}

cudaError_t sd_join_fast_redo(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 window, const u32* redo,
                              u32 n_redo, DevInfo* info, cudaStream_t st, i64* launches) {
    if (n_redo == 0) return cudaSuccess;
    JoinFastParams FP{};
    FP.j = jn_params(records, n_records, lay, cand, window, info);
    FP.j.win_lo = 0;
    FP.j.win_hi = window;
    FP.tiles = redo;
    FP.redo = nullptr;
    if (launches) ++*launches;
    return jn_k32(FP.j) ? jn_launch_fast<true>(FP, n_redo, true, st) : jn_launch_fast<false>(FP, n_redo, true, st);
}

cudaError_t sd_join(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 cand_cap, u64 win_lo, u64 win_hi,
                    int first_round, u64* tile_prefix, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = sd_join_tiles(n_records);
    if (tiles == 0) return cudaSuccess;
    constexpr size_t smem = sizeof(JoinSmem);
    cudaError_t e;
    if (first_round && (e = cudaMemsetAsync(&info->n_cand, 0, sizeof(u64), st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&info->win_end, 0, sizeof(u64), st)) != cudaSuccess) return e;
    JoinParams P = jn_params(records, n_records, lay, cand, cand_cap, info);
    P.win_lo = win_lo;
    P.win_hi = win_hi;
    P.first_round = first_round;
    P.tile_prefix = tile_prefix;
    k_join<<<(unsigned)tiles, JN_THREADS, smem, st>>>(P);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// ---- bucket join of the fused pipeline ------------------------------------------------------------
// buckets: nbuckets regions of `cap` records with counts cnt.  lay.sort_bits = the partitioned bits.
// info->n_cand = number of pairs written to cand[0 .. ); info->join_fallback != 0: they did not fit `window`.
int sd_join_bkt_max_cap() { return JB_STAGE_L; }
// the fused pipeline needs this many bits on top of every record of a bucket that are the same for the whole bucket
// (partitioned hash bits, or zeros above a narrowed hash): they carry the chain link
int sd_join_bkt_link_bits(u32 cap) { return cap <= (u32)JB_STAGE_S ? JB_NB_S : JB_NB_L; }

cudaError_t sd_join_bkt(const u64* buckets, u32* cnt, u32 cap, u32 nbuckets, const Layout& lay, u64* cand, u64 window,
                        int first_pass, int info_fresh, int prefer_small, int append, DevInfo* info, cudaStream_t st, i64* launches) {
    cudaError_t e = cudaSuccess;
    // (info_fresh: the whole status block was cleared for this call and nothing has counted pairs or raised a join flag yet)
    // append: info->n_cand keeps its value — the window already holds that many pairs of earlier chunks (S5: one flush per
    // full window, not per chunk) and the claims of this launch continue behind them
    if (!info_fresh && !append && (e = cudaMemsetAsync(&info->n_cand, 0, sizeof(u64), st)) != cudaSuccess) return e;
    static_assert(offsetof(DevInfo, nofit_inv) == offsetof(DevInfo, join_fallback) + 8, "cleared together");
    if (!info_fresh && (e = cudaMemsetAsync(&info->join_fallback, 0, 2 * sizeof(u32) + sizeof(u64), st)) != cudaSuccess) return e;  // and join_redo, nofit_inv
    if (nbuckets == 0) return cudaSuccess;
    JoinBktParams BP{};
    BP.j = jn_params(buckets, 0, lay, cand, window, info);
    BP.j.win_lo = 0;
    BP.j.win_hi = window;
    BP.j.first_round = first_pass;
    BP.cnt = cnt;
    BP.cap = cap;
    BP.nbuckets = nbuckets;
    // chain slot = the hash bits right below the partitioned ones (clamped to the hash field)
    const int top = lay.id_bits + lay.hash_bits;
    // prefer_small: the regions were sized for more records than they are expected to hold (the query filter of a cross-search
    // dropped most of them): the small instance takes every bucket it can stage and leaves the others open for a later call
    const bool small = cap <= (u32)JB_STAGE_S || prefer_small;
    BP.stage_cap = small ? std::min<u32>(cap, (u32)JB_STAGE_S) : cap;
    BP.j.slot_shift = std::max(lay.id_bits, top - lay.sort_bits - (small ? JB_SLOTB_S : JB_SLOTB_L));
    if (launches) ++*launches;
    const size_t smem = jb_smem_bytes(small, BP.stage_cap);
    if (small && !lay.cross) e = sd_launch_dep(k_join_bkt<JB_THREADS_S, JB_STAGE_S, JB_SLOTB_S, JB_NB_S, JB_MINB_S, false>, nbuckets, (unsigned)JB_THREADS_S, smem, st, BP);
    else if (small) e = sd_launch_dep(k_join_bkt<JB_THREADS_S, JB_STAGE_S, JB_SLOTB_S, JB_NB_S, JB_MINB_S, true>, nbuckets, (unsigned)JB_THREADS_S, smem, st, BP);
    else if (!lay.cross) e = sd_launch_dep(k_join_bkt<JB_THREADS_L, JB_STAGE_L, JB_SLOTB_L, JB_NB_L, JB_MINB_L, false>, nbuckets, (unsigned)JB_THREADS_L, smem, st, BP);
    else e = sd_launch_dep(k_join_bkt<JB_THREADS_L, JB_STAGE_L, JB_SLOTB_L, JB_NB_L, JB_MINB_L, true>, nbuckets, (unsigned)JB_THREADS_L, smem, st, BP);
    return e != cudaSuccess ? e : cudaGetLastError();
}
