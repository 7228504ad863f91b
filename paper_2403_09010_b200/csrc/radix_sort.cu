// radix_sort.cu — S2/K2: radix partition / LSD radix sort of 64-bit words, onesweep style.
//
// "Second, sort those tuples by the deletion variant.  This guarantees that all strings with
// matching deletion variants will be stored contiguously." (§I.B step 2; App. F.2
// step 2; App. F.3 step 2).  The paper's tools use a parallel CPU sort
// and a GPU merge sort.  Here equal variants only have to MEET, so the variant records are not
// sorted in full:
//   * fused pipeline (default): k_part2 splits each level-1 bin written by the generator on the next
//     hash bits into fixed-capacity buckets (one pass, no histogram, no look-back); the join compares
//     the remaining hash bits;
//   * exact pipeline (fallback): k_onesweep passes over the top `sort_bits` of the hash only, on exact
//     histograms that the generation kernel accumulates in its own pass;
//   * the packed candidate pair ids (S3b) and the merged survivors ARE sorted in full: k_histogram
//     (one read builds every digit place) + one k_onesweep per 8-bit digit.
// k_onesweep: each tile ranks its keys with per-warp shared-memory counters and peer masks, obtains
// its cross-tile exclusive prefix per digit by decoupled look-back over a status array (tile order =
// atomic ticket, so predecessors have always started), stages the tile in shared memory in digit
// order and writes each digit's keys to one contiguous global segment.
// Every pass reads n*8 and writes n*8 bytes: 16 B/word/pass of algorithmic traffic.
#include "kernels.h"

namespace {

// ---------------------------------------------------------------------------------------------
template <int THREADS>
__global__ void __launch_bounds__(THREADS) k_histogram(const u64* __restrict__ keys, u64 n, int begin_bit, int npass,
                                                      u32* __restrict__ ghist) {
    __shared__ u32 sh[8 * 256];
    for (int i = threadIdx.x; i < npass * 256; i += THREADS) sh[i] = 0;
    __syncthreads();
    const u64 stride = (u64)gridDim.x * THREADS;
    for (u64 i = (u64)blockIdx.x * THREADS + threadIdx.x; i < n; i += stride) {
        u64 k = keys[i];
        for (int p = 0; p < npass; ++p) atomicAdd(&sh[p * 256 + ((u32)(k >> (begin_bit + 8 * p)) & 255u)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < npass * 256; i += THREADS)
        if (sh[i]) atomicAdd(&ghist[i], sh[i]);
}

// exclusive scan of each pass's 256 bins, in place; one block of 256 threads per pass
__global__ void __launch_bounds__(256) k_hist_scan(u32* __restrict__ ghist) {
    sd_dep_wait();
    sd_dep_release();
    __shared__ u32 s_warp[9];
    u32* h = ghist + blockIdx.x * 256;
    u32 v = h[threadIdx.x], total;
    u32 e = sd_block_excl_sum<256>(v, &total, s_warp);
    h[threadIdx.x] = e;
}

// ---------------------------------------------------------------------------------------------
// S3b, first half: duplicate suppression BEFORE the sort (k_cand_filter).  A pair within distance d shares several
// deletion variants, so the join emits it several times (config 3: 3.67 M candidates for 0.52 M distinct pairs; the
// paper's real repertoires: 137 M matched for 56 M unique).  Instead of sorting all of them, every
// candidate is first offered to an open-addressing hash set of packed pair ids (64-bit compare-and-swap, linear
// probing, a few probes at most): a candidate that finds ITSELF in the set is dropped, one that claims an empty slot
// or finds no room after the probe limit is kept.  The set is best effort by design — a full table only lets
// duplicates through — because the sorted candidates are still compared with their left neighbour in the verifier:
// the result cannot depend on it.  The kept candidates are compacted (block scan, one global atomic per tile) and
// their digit histograms for the LSD passes are accumulated in the same sweep: this kernel replaces k_histogram on the
// candidate side.  Table entries hold key + 1 (0 = empty).
constexpr int CF_THREADS = 256, CF_IPT = 8, CF_TILE = CF_THREADS * CF_IPT, CF_PROBES = 6;

__global__ void __launch_bounds__(CF_THREADS) k_cand_filter(const u64* __restrict__ cand, u64 n, unsigned long long* __restrict__ table,
                                                           int table_bits, u64* __restrict__ out, u64* n_out, int npass,
                                                           u32* __restrict__ ghist) {
    __shared__ u32 sh[8 * 256];
    __shared__ u32 s_warp[CF_THREADS / 32 + 1];
    __shared__ u64 s_base;
    const u32 tid = threadIdx.x;
    for (int i = tid; i < npass * 256; i += CF_THREADS) sh[i] = 0;
    const u64 base = (u64)blockIdx.x * CF_TILE;
    const u64 tmask = (1ull << table_bits) - 1ull;
    u64 key[CF_IPT];
    u32 keep = 0;
#pragma unroll
    for (int k = 0; k < CF_IPT; ++k) {
        const u64 pos = base + (u64)k * CF_THREADS + tid;
        key[k] = pos < n ? cand[pos] : 0ull;
    }
#pragma unroll
    for (int k = 0; k < CF_IPT; ++k) {
        const u64 pos = base + (u64)k * CF_THREADS + tid;
        if (pos < n) {
            const unsigned long long want = key[k] + 1ull;
            u64 h = (key[k] * 0x9e3779b97f4a7c15ull) >> (64 - table_bits);
            bool dup = false;
            for (int pr = 0; pr < CF_PROBES; ++pr) {
                const unsigned long long old = atomicCAS(&table[h], 0ull, want);
                if (old == 0ull) break;  // claimed: first time this pair is seen
                if (old == want) {
                    dup = true;
                    break;
                }
                h = (h + 1) & tmask;
            }
            if (!dup) keep |= 1u << k;
        }
    }
    __syncthreads();  // sh cleared
    u32 total;
    const u32 rank = sd_block_excl_sum<CF_THREADS>(__popc(keep), &total, s_warp);
    if (tid == 0) s_base = total ? (u64)atomicAdd((unsigned long long*)n_out, (unsigned long long)total) : 0ull;
    __syncthreads();
    u64 at = s_base + rank;
#pragma unroll
    for (int k = 0; k < CF_IPT; ++k)
        if ((keep >> k) & 1u) {
            out[at++] = key[k];
            for (int p = 0; p < npass; ++p) atomicAdd(&sh[p * 256 + ((u32)(key[k] >> (8 * p)) & 255u)], 1u);
        }
    __syncthreads();
    for (int i = tid; i < npass * 256; i += CF_THREADS)
        if (sh[i]) atomicAdd(&ghist[i], sh[i]);
}

// ---------------------------------------------------------------------------------------------
#define OS_FLAG_AGG (1u << 30)
#define OS_FLAG_PRE (2u << 30)
#define OS_MASK ((1u << 30) - 1)
constexpr int OS_LB = 4;  // look-back: predecessors inspected per round trip

// Shared tail of both tile paths: per-digit decoupled look-back, then the coalesced write-out of the
// tile staged in digit order.  `total` / `tstart` (threads < 256): this tile's count and tile-local
// start of digit tid.  The aggregate was published by the caller.
template <int THREADS, int IPT, bool FULLT>
__device__ __forceinline__ void os_lookback_and_write(u64* __restrict__ out, const u32 tile_n, const u32 tile, const int shift,
                                                      const u32* __restrict__ gbase, u32* st, const u32 total,
                                                      const u32 tstart, const u64* skeys, u32* s_gofs, const bool claim,
                                                      const u32 claimed) {
    const u32 tid = threadIdx.x;
    if (claim) {
        if (tid < 256) s_gofs[tid] = claimed - tstart;
    } else if (tid < 256) {
        u32 excl = 0;
        if (tile != 0) {
            // OS_LB predecessors per round trip: the walk back to the nearest inclusive prefix is a chain
            // of L2 latencies, so loads are issued in batches and consumed in order
            const u32* p = st;
            u32 rem = tile;
            bool done = false;
            while (!done) {
                u32 sv[OS_LB];
#pragma unroll
                for (int j = 0; j < OS_LB; ++j) sv[j] = ((u32)j < rem) ? sd_ld_relaxed32(p - 256 * (j + 1)) : OS_FLAG_PRE;
                int used = 0;
#pragma unroll
                for (int j = 0; j < OS_LB; ++j) {
                    if (!done && used == j) {
                        const u32 f = sv[j] >> 30;
                        if (f != 0) {
                            excl += sv[j] & OS_MASK;
                            used = j + 1;
                            done = (f == 2);
                        }
                    }
                }
                p -= 256 * used;
                rem -= (u32)used;
            }
            sd_st_relaxed32(st, OS_FLAG_PRE | (excl + total));
        }
        s_gofs[tid] = gbase[tid] + excl - tstart;
    }
    __syncthreads();

    // ---- write out: consecutive threads -> consecutive slots of one digit's global segment ----
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const u32 pos = tid + k * THREADS;
        if (FULLT || pos < tile_n) {
            const u64 kk = skeys[pos];
            out[s_gofs[(u32)(kk >> shift) & 255u] + pos] = kk;
        }
    }
}

// ---- stable tile: ties keep their input order (what every LSD pass after the first needs when the
//      tile mixes several values of the digits already sorted) ----
template <int THREADS, int IPT, bool FULLT>
__device__ __forceinline__ void os_tile(const u64 (&key)[IPT], u64* __restrict__ out, const u32 tile_n, const u32 tile,
                                        const int shift, const u32* __restrict__ gbase, u32* __restrict__ status,
                                        u64* skeys, u32* whist, u32* wmask, u32* s_gofs, u32* s_warp) {
    constexpr int NW = THREADS / 32;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 wbase = warp * (32 * IPT);
    const u32 lane_lt = (1u << lane) - 1u;

    // ---- early counts: per-warp digit histograms by shared-memory atomics ----
    u32* myhist = whist + warp * 256;
#pragma unroll
    for (int k = 0; k < IPT; ++k)
        if (FULLT || (wbase + 32 * k + lane) < tile_n) atomicAdd(&myhist[(u32)(key[k] >> shift) & 255u], 1u);
    __syncthreads();

    // ---- per digit: exclusive offsets across warps, tile total; publish the aggregate EARLY so that
    //      successors never wait on this tile's ranking ----
    u32 total = 0;
    u32* st = status + (u64)tile * 256 + tid;
    if (tid < 256) {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const u32 c = whist[w * 256 + tid];
            whist[w * 256 + tid] = total;
            total += c;
        }
        sd_st_relaxed32(st, (tile == 0 ? OS_FLAG_PRE : OS_FLAG_AGG) | total);
    }
    u32 tile_sum;
    const u32 tstart = sd_block_excl_sum<THREADS>(total, &tile_sum, s_warp);
    if (tid < 256) {
#pragma unroll
        for (int w = 0; w < NW; ++w) whist[w * 256 + tid] += tstart;  // now: next free slot of (warp, digit)
    }
    __syncthreads();

    // ---- rank inside the warp's chunk (stable: position order = (k, lane)) and stage in digit order ----
    // peer mask by one shared-memory atomic OR per key (measured 2.5x cheaper than 8 ballots on sm_100a)
    u32* mymask = wmask + warp * 256;
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const bool valid = FULLT || (wbase + 32 * k + lane) < tile_n;
        const u32 dg = (u32)(key[k] >> shift) & 255u;
        if (valid) atomicOr(&mymask[dg], 1u << lane);
        __syncwarp();
        const u32 peers = mymask[dg];
        const u32 pre = myhist[dg];
        __syncwarp();
        const u32 below = __popc(peers & lane_lt);
        if (valid && below == 0) {
            myhist[dg] = pre + __popc(peers);
            mymask[dg] = 0;
        }
        __syncwarp();
        if (valid) skeys[pre + below] = key[k];
    }
    os_lookback_and_write<THREADS, IPT, FULLT>(out, tile_n, tile, shift, gbase, st, total, tstart, skeys, s_gofs, false, 0u);
}

// ---- grouping tile: ties land in arbitrary order.  Legal for the first pass of a keys-only sort and
//      for any later pass over a tile whose keys agree on every digit already sorted (then any order
//      inside the tile is a sorted order).  One shared-memory atomic per key returns its rank inside
//      (tile, digit): no peer masks, no per-warp counters. ----
template <int THREADS, int IPT, bool FULLT>
__device__ __forceinline__ void os_tile_group(const u64 (&key)[IPT], u64* __restrict__ out, const u32 tile_n, const u32 tile,
                                              const int shift, u32* __restrict__ gbase, u32* __restrict__ status,
                                              u64* skeys, u32* bhist, u32* s_gofs, u32* s_warp, const bool claim) {
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 wbase = warp * (32 * IPT);
    u32 rank[IPT / 2];  // two 16-bit ranks per word (a tile holds < 65536 keys)
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        u32 r = 0;
        if (FULLT || (wbase + 32 * k + lane) < tile_n) r = atomicAdd(&bhist[(u32)(key[k] >> shift) & 255u], 1u);
        if (k & 1) rank[k >> 1] |= r << 16;
        else rank[k >> 1] = r;
    }
    __syncthreads();
    u32 total = 0;
    u32* st = status + (u64)tile * 256 + tid;
    u32 claimed = 0;
    if (tid < 256) {
        total = bhist[tid];
        // claim mode (first pass of a keys-only sort: no order to keep between tiles either): the tile takes
        // its slice of every digit's output range with one atomic on the running bin base — no status row,
        // no look-back; the round trip overlaps the scan and the staging below
        if (claim) claimed = total ? atomicAdd(&gbase[tid], total) : 0u;
        else sd_st_relaxed32(st, (tile == 0 ? OS_FLAG_PRE : OS_FLAG_AGG) | total);
    }
    u32 tile_sum;
    const u32 tstart = sd_block_excl_sum<THREADS>(total, &tile_sum, s_warp);
    if (tid < 256) bhist[tid] = tstart;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        if (FULLT || (wbase + 32 * k + lane) < tile_n) {
            const u32 r = (k & 1) ? (rank[k >> 1] >> 16) : (rank[k >> 1] & 0xffffu);
            skeys[bhist[(u32)(key[k] >> shift) & 255u] + r] = key[k];
        }
    }
    os_lookback_and_write<THREADS, IPT, FULLT>(out, tile_n, tile, shift, gbase, st, total, tstart, skeys, s_gofs, claim, claimed);
}

// smask: the bits whose order the pass must preserve.  ~0 = stable sort (every tile takes the stable
// path).  Otherwise the input is sorted on the bits of smask (the digits already processed) and ties
// may land in any order: a tile whose first and last key agree on smask holds one value of those bits
// and takes the grouping path.  smask == 0 (first pass): claim mode, tile = block index.
template <int THREADS, int IPT, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) k_onesweep(const u64* __restrict__ in, u64* __restrict__ out, u32 n, int shift,
                                                           u64 smask, u32* __restrict__ gbase, u32* __restrict__ status,
                                                           u32* __restrict__ ticket, const u64* __restrict__ n_dev) {
    static_assert(IPT % 2 == 0 && THREADS * IPT < 65536, "rank packing");
    constexpr int TILE = THREADS * IPT, NW = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* skeys = reinterpret_cast<u64*>(smem_raw);      // TILE keys, digit order
    u32* whist = reinterpret_cast<u32*>(skeys + TILE);  // NW x 256 per-warp digit counters / slot pointers
    u32* wmask = whist + NW * 256;                      // NW x 256 per-warp peer masks (stable path)
    u32* s_gofs = wmask + NW * 256;                     // 256: global offset of digit d minus its tile start
    __shared__ u32 s_tile;
    __shared__ u32 s_warp[NW + 1];
    __shared__ u64 s_ends[2];

    sd_dep_wait();  // (the passes are launched as dependents of one another)
    sd_dep_release();
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool claim = smask == 0;
    // n_dev: the key count lives on the device (the grid was sized for an upper bound: surplus blocks leave at once —
    // tiles are numbered by ticket, so no working tile ever waits on one of them)
    if (n_dev) n = (u32)*n_dev;
    if (!claim && tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < (claim ? 256 : 2 * NW * 256); i += THREADS) whist[i] = 0;
    __syncthreads();
    const u32 tile = claim ? blockIdx.x : s_tile;
    const u32 base = tile * TILE;
    if (base >= n) return;  // (block-uniform)
    const u32 tile_n = min((u32)TILE, n - base);
    const bool full = tile_n == (u32)TILE;

    // ---- load, warp-striped: item k of lane l is tile position wbase + 32k + l (coalesced) ----
    const u32 wbase = warp * (32 * IPT);
    u64 key[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const u32 pos = wbase + 32 * k + lane;
        key[k] = (full || pos < tile_n) ? in[base + pos] : ~0ull;
    }
    bool group = claim;
    if (!claim && smask != ~0ull && full) {  // block-uniform
        if (tid == 0) s_ends[0] = key[0];
        if (tid == THREADS - 1) s_ends[1] = key[IPT - 1];
        __syncthreads();
        group = ((s_ends[0] ^ s_ends[1]) & smask) == 0;
    }
    if (group && full)
        os_tile_group<THREADS, IPT, true>(key, out, tile_n, tile, shift, gbase, status, skeys, whist, s_gofs, s_warp, claim);
    else if (group)
        os_tile_group<THREADS, IPT, false>(key, out, tile_n, tile, shift, gbase, status, skeys, whist, s_gofs, s_warp, claim);
    else if (full)
        os_tile<THREADS, IPT, true>(key, out, tile_n, tile, shift, gbase, status, skeys, whist, wmask, s_gofs, s_warp);
    else
        os_tile<THREADS, IPT, false>(key, out, tile_n, tile, shift, gbase, status, skeys, whist, wmask, s_gofs, s_warp);
}

// ---------------------------------------------------------------------------------------------
// Level-2 partition of the fused pipeline (k_part2).  Input: 256 level-1 bins of capacity cap1 with
// their record counts cnt1 (written by k_gen2_part).  A tile of a bin is split on the next b2 hash bits
// into that bin's 2^b2 BUCKETS, each a fixed-capacity region of cap2 records: bucket (bin, digit) lives
// at ((bin << b2) + digit) * cap2 and cnt2 counts what it holds.  This is the grouping tile of
// k_onesweep in claim mode — one shared-memory atomic per key returns its rank inside (tile, digit), one
// global atomic per digit claims the tile's slice of the bucket, the tile leaves staged in digit order
// — without histograms, tickets or look-back, because nothing downstream needs the records of a bucket
// contiguous with the next bucket or in any order.  A bucket that would overflow raises
// info->part_overflow (the host falls back to the exact pipeline).
constexpr int P2_THREADS = 256, P2_IPT = 16, P2_MINB = 4, P2_TILE = P2_THREADS * P2_IPT;  // (tiles of 12 / 20 / 24 keys per thread: within 2 %)

struct Part2Params {
    const u64* bins;
    const u32* cnt1;
    u64 cap1;
    u64* buckets;
    u32* cnt2;
    u32 cap2;
    int b2, shift;  // digit = (record >> shift) & (2^b2 - 1)
    u32 tiles_per_bin;
    DevInfo* info;
    // query filter (cross-search, FILT instance): a record of set B is kept only if some record of set A of the same bin has
    // the same fbits hash bits below the bin digit; the first cnt_a[bin] records of a bin are set A's (generated first)
    const u32* bitmap;  // 256 bitmaps of 2^fbits bits
    const u32* cnt_a;
    int fbits, fshift;
};

// One tile of k_part2 from the ranking on: `key` / `valid` (bit k: key[k] takes part; FULL: all of them) in registers.
template <bool FULL>
__device__ __forceinline__ void p2_tile(const Part2Params& P, const u64 (&key)[P2_IPT], const u32 valid, const u32 n_valid, const u32 bin,
                                        u64* skeys, u32* bhist, u32* s_gofs, u32* s_warp) {
    const u32 tid = threadIdx.x;
    const u32 dmask = (1u << P.b2) - 1u;
    u32 rank[P2_IPT / 2];  // two 16-bit ranks per word
#pragma unroll
    for (int k = 0; k < P2_IPT; ++k) {
        u32 r = 0;
        if (FULL || ((valid >> k) & 1u)) r = atomicAdd(&bhist[(u32)(key[k] >> P.shift) & dmask], 1u);
        if (k & 1) rank[k >> 1] |= r << 16;
        else rank[k >> 1] = r;
    }
    __syncthreads();
    const u32 total = bhist[tid];
    u32 claimed = 0;
    bool dead = false;
    if (total) claimed = atomicAdd(&P.cnt2[(bin << P.b2) + tid], total);
    u32 tile_sum;
    const u32 tstart = sd_block_excl_sum<P2_THREADS>(total, &tile_sum, s_warp);
    bhist[tid] = tstart;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < P2_IPT; ++k) {
        if (FULL || ((valid >> k) & 1u)) {
            const u32 r = (k & 1) ? (rank[k >> 1] >> 16) : (rank[k >> 1] & 0xffffu);
            skeys[bhist[(u32)(key[k] >> P.shift) & dmask] + r] = key[k];
        }
    }
    // the claim is looked at only now: its round trip to L2 ran under the scan and the staging stores
    if (total && claimed + total > P.cap2) {
        atomicOr(&P.info->part_overflow, 2u);
        dead = true;
    }
    s_gofs[tid] = dead ? 0xffffffffu : ((bin << P.b2) + tid) * P.cap2 + claimed - tstart;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < P2_IPT; ++k) {
        const u32 pos = tid + k * P2_THREADS;
        if (FULL || pos < n_valid) {
            const u64 kk = skeys[pos];
            const u32 g = s_gofs[(u32)(kk >> P.shift) & dmask];
            if (g != 0xffffffffu) P.buckets[g + pos] = kk;
        }
    }
}

__global__ void __launch_bounds__(P2_THREADS, P2_MINB) k_part2(const Part2Params P) {
    sd_dep_wait();  // (launched as a dependent of the generator)
    sd_dep_release();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* skeys = reinterpret_cast<u64*>(smem_raw);
    __shared__ u32 bhist[256];
    __shared__ u32 s_gofs[256];
    __shared__ u32 s_warp[P2_THREADS / 32 + 1];
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 bin = blockIdx.x / P.tiles_per_bin, k0 = blockIdx.x % P.tiles_per_bin;
    const u32 n_bin = (u32)min((u64)P.cnt1[bin], P.cap1);
    const u32 base = k0 * P2_TILE;
    if (base >= n_bin) return;
    const u32 tile_n = min((u32)P2_TILE, n_bin - base);
    const u64* in = P.bins + (u64)bin * P.cap1 + base;
    bhist[tid] = 0;
    const u32 wbase = warp * (32 * P2_IPT);
    u64 key[P2_IPT];
    if (tile_n == (u32)P2_TILE) {  // (block-uniform)
#pragma unroll
        for (int k = 0; k < P2_IPT; ++k) key[k] = in[wbase + 32 * k + lane];
        __syncthreads();
        p2_tile<true>(P, key, 0xffffffffu, tile_n, bin, skeys, bhist, s_gofs, s_warp);
    } else {
        u32 valid = 0;
#pragma unroll
        for (int k = 0; k < P2_IPT; ++k) {
            const u32 pos = wbase + 32 * k + lane;
            const bool ok = pos < tile_n;
            key[k] = ok ? in[pos] : 0ull;
            valid |= (ok ? 1u : 0u) << k;
        }
        __syncthreads();
        p2_tile<false>(P, key, valid, tile_n, bin, skeys, bhist, s_gofs, s_warp);
    }
}

// The filtering form (cross-search, see k_bin_bitmap below): a block walks P2F_TILES consecutive tiles of one bin with the
// bin's bitmap in shared memory, keeps what passes in a staging tile (one slice per warp), and partitions the staging tile
// whenever the next input tile might not fit — most set-B records never reach the ranking, the scatter or HBM again.
constexpr int P2F_TILES = 16, P2F_IPT = 8, P2F_IN = P2_THREADS * P2F_IPT;
__global__ void __launch_bounds__(P2_THREADS, 2) k_part2f(const Part2Params P) {
    sd_dep_wait();
    sd_dep_release();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* skeys = reinterpret_cast<u64*>(smem_raw);       // staging tile / digit-ordered tile
    u32* sbm = reinterpret_cast<u32*>(skeys + P2_TILE);  // this bin's bitmap
    __shared__ u32 bhist[256];
    __shared__ u32 s_gofs[256];
    __shared__ u32 s_warp[P2_THREADS / 32 + 1];
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 groups = (P.tiles_per_bin + P2F_TILES - 1) / P2F_TILES;
    const u32 bin = blockIdx.x / groups, t0 = (blockIdx.x % groups) * P2F_TILES;
    const u32 n_bin = (u32)min((u64)P.cnt1[bin], P.cap1);
    if (t0 * P2_TILE >= n_bin) return;
    {
        const u32 words = 1u << (P.fbits - 5);
        const uint4* src = reinterpret_cast<const uint4*>(P.bitmap + (size_t)bin * words);
        for (u32 i = tid; i < words / 4; i += P2_THREADS) reinterpret_cast<uint4*>(sbm)[i] = src[i];
    }
    const u32 na = P.cnt_a[bin], fmask = (1u << P.fbits) - 1u;
    // Staging: every warp keeps what passes in its own slice of the staging tile (ballot + popcount, no block-wide step);
    // the block partitions the tile when some warp's slice could not take another input tile.
    constexpr u32 SLICE = P2_TILE / (P2_THREADS / 32);  // 512 slots per warp
    static_assert(SLICE >= 2 * 32 * P2F_IPT, "a slice takes at least two input tiles of its warp");
    __shared__ u32 s_wcnt[P2_THREADS / 32];
    if (tid < P2_THREADS / 32) s_wcnt[tid] = 0;
    u32 wcnt = 0;  // records in this warp's slice (warp-uniform)
    auto flush = [&]() {  // partitions the staging tile (called by all threads)
        if (lane == 0) s_wcnt[warp] = wcnt;
        __syncthreads();
        u64 key[P2_IPT];
        u32 valid = 0, n_stage = 0;
#pragma unroll
        for (int w = 0; w < P2_THREADS / 32; ++w) n_stage += s_wcnt[w];
#pragma unroll
        for (int k = 0; k < P2_IPT; ++k) {
            const u32 pos = tid + k * P2_THREADS;
            const bool ok = (pos % SLICE) < s_wcnt[pos / SLICE];
            key[k] = ok ? skeys[pos] : 0ull;
            valid |= (ok ? 1u : 0u) << k;
        }
        bhist[tid] = 0;
        __syncthreads();  // staging tile read by everyone, histogram cleared
        p2_tile<false>(P, key, valid, n_stage, bin, skeys, bhist, s_gofs, s_warp);
        __syncthreads();  // skeys free again
        wcnt = 0;
    };
    __syncthreads();  // bitmap loaded
    // input in tiles of P2F_IPT keys per thread, the next tile's loads in flight while this one is tested and appended
    const u32 r0 = t0 * P2_TILE, r1 = min(n_bin, (t0 + P2F_TILES) * (u32)P2_TILE);
    const u64* in = P.bins + (u64)bin * P.cap1;
    const u32 fw = warp * (32 * P2F_IPT);
    const u32 lane_lt = (1u << lane) - 1u;
    u64* const slice = skeys + warp * SLICE;
    u64 nxt[P2F_IPT];
#pragma unroll
    for (int k = 0; k < P2F_IPT; ++k) {
        const u32 pos = r0 + fw + 32 * k + lane;
        nxt[k] = pos < r1 ? in[pos] : 0ull;
    }
    for (u32 base = r0; base < r1; base += P2F_IN) {
        u64 key[P2F_IPT];
#pragma unroll
        for (int k = 0; k < P2F_IPT; ++k) key[k] = nxt[k];
#pragma unroll
        for (int k = 0; k < P2F_IPT; ++k) {
            const u32 pos = base + P2F_IN + fw + 32 * k + lane;
            nxt[k] = pos < r1 ? in[pos] : 0ull;
        }
        // could this tile overflow a slice?  (one barrier per input tile, and only this one)
        if (__syncthreads_or(wcnt + 32 * P2F_IPT > SLICE)) flush();
#pragma unroll
        for (int k = 0; k < P2F_IPT; ++k) {
            const u32 pos = base + fw + 32 * k + lane;
            bool keep = false;
            if (pos < r1) {
                const u32 idx = (u32)(key[k] >> P.fshift) & fmask;
                keep = pos < na || ((sbm[idx >> 5] >> (idx & 31u)) & 1u);
            }
            const u32 bal = __ballot_sync(SD_FULL, keep);
            if (keep) slice[wcnt + __popc(bal & lane_lt)] = key[k];
            wcnt += __popc(bal);
        }
    }
    flush();
}


// Query filter of a cross-search (reading the paper's asymmetric use, "both the query and reference sets", with
// a small query set): one block per level-1 bin marks, for the set-A records of the bin (its first cnt_a[bin] records: set A
// is generated first), the fbits hash bits below the bin digit.  k_part2f then drops every set-B record whose bits are
// not marked: no record of set A can have its hash, so it cannot make a pair — the result is unchanged.
constexpr int BM_THREADS = 512;
__global__ void __launch_bounds__(BM_THREADS) k_bin_bitmap(const u64* __restrict__ bins, const u32* __restrict__ cnt_a, u64 cap1,
                                                          u32* __restrict__ bitmap, int fbits, int fshift) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u32* sb = reinterpret_cast<u32*>(smem_raw);
    const u32 bin = blockIdx.x, words = 1u << (fbits - 5), fmask = (1u << fbits) - 1u;
    for (u32 i = threadIdx.x; i < words; i += BM_THREADS) sb[i] = 0;
    __syncthreads();
    const u32 n = (u32)min((u64)cnt_a[bin], cap1);
    const u64* in = bins + (u64)bin * cap1;
    for (u32 i = threadIdx.x; i < n; i += BM_THREADS) {
        const u32 idx = (u32)(in[i] >> fshift) & fmask;
        atomicOr(&sb[idx >> 5], 1u << (idx & 31u));
    }
    __syncthreads();
    for (u32 i = threadIdx.x; i < words; i += BM_THREADS) bitmap[(size_t)bin * words + i] = sb[i];
}

struct OsVariant {
    int threads, ipt;
    size_t smem;
    void (*kernel)(const u64*, u64*, u32, int, u64, u32*, u32*, u32*, const u64*);
};
template <int THREADS, int IPT, int MINB>
constexpr OsVariant os_variant() {
    return {THREADS, IPT, (size_t)THREADS * IPT * 8 + 2 * (THREADS / 32) * 256 * 4 + 256 * 4, k_onesweep<THREADS, IPT, MINB>};
}
// Tile shapes.  [0] is the one the pipeline uses (round 1 swept 17 shapes on config 3: 256 x 16 with four
// resident blocks was the fastest pass, 3.6 TB/s; 512 x 16 and 384 x 18 within 3 %); the others stay
// selectable per context (SYMDEL_OPT_SORT_VARIANT) so that the parity tests cover other tile geometries.
const OsVariant OS_VARIANTS[] = {os_variant<256, 16, 4>(), os_variant<512, 16, 2>(), os_variant<384, 18, 2>(),
                                 os_variant<256, 12, 4>()};
constexpr int OS_NVARIANTS = sizeof(OS_VARIANTS) / sizeof(OS_VARIANTS[0]);
constexpr int OS_MIN_TILE = 256 * 12;  // scratch is sized for the smallest tile of any variant

}  // namespace

// ---------------------------------------------------------------------------------------------
i64 sd_sort_tiles(i64 n) { return (n + OS_MIN_TILE - 1) / OS_MIN_TILE; }

int sd_sort_variants() { return OS_NVARIANTS; }

// Per-device state of this translation unit (dynamic shared-memory limits): set for the current device by every
// symdel_create.
cudaError_t sd_sort_setup() {
    cudaError_t e;
    for (int v = 0; v < OS_NVARIANTS; ++v)
        if ((e = cudaFuncSetAttribute(OS_VARIANTS[v].kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)OS_VARIANTS[v].smem)) != cudaSuccess)
            return e;
    if ((e = cudaFuncSetAttribute(k_part2f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P2_TILE * 8 + (size_t)(1 << SD_FBITS_MAX) / 8))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_bin_bitmap, cudaFuncAttributeMaxDynamicSharedMemorySize, (1 << SD_FBITS_MAX) / 8)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_part2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P2_TILE * 8));
}

// scratch layout: [npass][256] u32 histograms | [npass] tickets (padded to 256 B) | [npass][tiles][256] u32 status
i64 sd_sort_scratch_bytes(i64 n, int npass) {
    return (i64)npass * 256 * 4 + 256 + (i64)npass * sd_sort_tiles(n) * 256 * 4;
}

// Zeroes the scratch (histograms, tickets, status).  Call before the histograms are accumulated.
cudaError_t sd_sort_prepare(void* scratch, i64 n, int npass, cudaStream_t st) {
    return cudaMemsetAsync(scratch, 0, (size_t)sd_sort_scratch_bytes(n, npass), st);
}

u32* sd_sort_hist_ptr(void* scratch) { return reinterpret_cast<u32*>(scratch); }

cudaError_t sd_sort_histogram(const u64* keys, i64 n, int begin_bit, int npass, void* scratch, cudaStream_t st,
                              i64* launches) {
    if (n == 0) return cudaSuccess;
    int blocks = (int)std::min<i64>((n + 255) / 256, 148 * 8);
    k_histogram<256><<<blocks, 256, 0, st>>>(keys, (u64)n, begin_bit, npass, sd_sort_hist_ptr(scratch));
    if (launches) ++*launches;
    return cudaGetLastError();
}

// Candidate filter + histograms (see k_cand_filter).  table: 2^table_bits zeroed 64-bit slots; *n_out (device) is
// cleared here and receives the number of candidates kept in out[0 .. ).  The histograms go to `scratch` as with
// sd_sort_histogram (bits [0, 8 * npass) of the keys).
cudaError_t sd_cand_filter(const u64* cand, i64 n, void* table, int table_bits, u64* out, u64* n_out, int npass, void* scratch,
                           cudaStream_t st, i64* launches) {
    cudaError_t e = cudaMemsetAsync(n_out, 0, sizeof(u64), st);
    if (e != cudaSuccess || n == 0) return e;
    const unsigned blocks = (unsigned)((n + CF_TILE - 1) / CF_TILE);
    k_cand_filter<<<blocks, CF_THREADS, 0, st>>>(cand, (u64)n, (unsigned long long*)table, table_bits, out, n_out, npass,
                                                sd_sort_hist_ptr(scratch));
    if (launches) ++*launches;
    return cudaGetLastError();
}

// Turns the raw per-digit counts into exclusive bin bases (one tiny launch).
cudaError_t sd_sort_hist_scan(void* scratch, int npass, cudaStream_t st, i64* launches) {
    if (npass == 0) return cudaSuccess;
    if (sd_launch_dep(k_hist_scan, (unsigned)npass, 256u, 0, st, sd_sort_hist_ptr(scratch)) != cudaSuccess) return cudaGetLastError();
    if (launches) ++*launches;
    return cudaGetLastError();
}

// Runs the passes.  The histograms in `scratch` must hold exclusive bin bases (sd_sort_hist_scan).
// n_dev != nullptr: the number of keys is *n_dev (device memory), n is only an upper bound that sizes the grids.
// Returns in *result the buffer (keys or tmp) that holds the sorted records.
// stable = 1: ties keep their input order.  stable = 0: keys-only sort, ties in arbitrary order (lets
// uniform tiles take the cheaper grouping path).
cudaError_t sd_sort_passes(u64* keys, u64* tmp, i64 n, const u64* n_dev, int begin_bit, int npass, int stable, int variant,
                           void* scratch, cudaStream_t st, u64** result, i64* launches) {
    *result = keys;
    if (n == 0 || npass == 0) return cudaSuccess;
    const OsVariant& V = OS_VARIANTS[variant >= 0 && variant < OS_NVARIANTS ? variant : 0];
    u32* hist = sd_sort_hist_ptr(scratch);
    u32* tickets = hist + npass * 256;
    u32* status = tickets + 64;
    const i64 tile = (i64)V.threads * V.ipt;
    const i64 tiles = (n + tile - 1) / tile;
    const i64 status_stride = sd_sort_tiles(n) * 256;
    u64 *src = keys, *dst = tmp;
    for (int p = 0; p < npass; ++p) {
        const u64 smask = stable ? ~0ull : (((1ull << (8 * p)) - 1ull) << begin_bit);
        const cudaError_t e = sd_launch_dep(V.kernel, (unsigned)tiles, (unsigned)V.threads, V.smem, st, (const u64*)src, dst, (u32)n, begin_bit + 8 * p,
                                            smask, hist + p * 256, status + (size_t)p * status_stride, tickets + p, n_dev);
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
        std::swap(src, dst);
    }
    *result = src;
    return cudaGetLastError();
}

// Level-2 partition of the fused pipeline: bins (256 x cap1, counts cnt1) -> buckets (2^(8+b2) x cap2,
// counts cnt2, zeroed here).  shift = bit of the record where the b2-bit digit starts.  b2 == 0: no-op
// for the caller (the bins are the buckets).
cudaError_t sd_bin_bitmap(const u64* bins, const u32* cnt_a, i64 cap1, u32* bitmap, int fbits, int fshift, cudaStream_t st, i64* launches) {
    k_bin_bitmap<<<256, BM_THREADS, (size_t)(1 << fbits) / 8, st>>>(bins, cnt_a, (u64)cap1, bitmap, fbits, fshift);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_part2(const u64* bins, const u32* cnt1, i64 cap1, u64* buckets, u32* cnt2, i64 cap2, int b2, int shift,
                     int counts_cleared, const u32* bitmap, const u32* cnt_a, int fbits, int fshift, DevInfo* info, cudaStream_t st,
                     i64* launches) {
    cudaError_t e;
    const size_t smem = (size_t)P2_TILE * 8 + (bitmap ? (size_t)(1 << fbits) / 8 : 0);
    if (!counts_cleared && (e = cudaMemsetAsync(cnt2, 0, ((size_t)256 << b2) * sizeof(u32), st)) != cudaSuccess) return e;
    Part2Params P{};
    P.bins = bins;
    P.cnt1 = cnt1;
    P.cap1 = (u64)cap1;
    P.buckets = buckets;
    P.cnt2 = cnt2;
    P.cap2 = (u32)cap2;
    P.b2 = b2;
    P.shift = shift;
    P.tiles_per_bin = (u32)((cap1 + P2_TILE - 1) / P2_TILE);
    P.info = info;
    P.bitmap = bitmap;
    P.cnt_a = cnt_a;
    P.fbits = fbits;
    P.fshift = fshift;
    if (bitmap) e = sd_launch_dep(k_part2f, 256 * ((P.tiles_per_bin + P2F_TILES - 1) / P2F_TILES), (unsigned)P2_THREADS, smem, st, P);
    else e = sd_launch_dep(k_part2, 256 * P.tiles_per_bin, (unsigned)P2_THREADS, smem, st, P);
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    return cudaGetLastError();
}
