// emit.cu — S3a/K3: run boundaries and candidate-pair emission over the sorted records.
//
// "Use the sorted array to identify groups of input strings that generate identical deletion
// variants, and transform this to an array of neighbor candidates" (App. F.2 step 3);
// "For each group v_g, generate all possible matching sequence pairs {(i', i'')} within the group"
// (App. F.3 step 3); a variant shared by m sequences yields m(m-1)/2 pairs
// (PAPER.md:96).  Output slots are allocated by prefix sums before anything is written
// ("avoid race condition by preallocating the outputs", Fig. S8).
//
// Record t pairs with the EARLIER records of its run: partner range [a(t), b(t)).
//   self : [run_start(t), t)
//   cross: records are sorted by (hash, id) and query ids are below reference ids, so a run is
//          [q .. q r .. r]; a reference record pairs with [run_start, first reference of the run),
//          a query record with nothing.
// The per-record counts are scanned inside the tile; a tile claims its output range with one atomic
// add (candidate order is irrelevant: they are sorted next); pairs are then written by FLAT pair index (binary search into the scanned counts), so a
// long run is spread over the whole block instead of serialising one thread.  Only pairs whose flat
// index lies in [win_lo, win_hi) are written: when the candidate buffer is smaller than the total,
// the host replays the kernel once per window (later rounds reuse the saved tile prefixes).
#include "kernels.h"

namespace {

constexpr int EM_THREADS = 256, EM_IPT = 4, EM_TILE = EM_THREADS * EM_IPT;

__device__ __forceinline__ u64 block_excl_sum64(u64 v, u64* total, u64* s_warp /* [EM_THREADS/32 + 1] */) {
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u64 inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u64 t = __shfl_up_sync(SD_FULL, inc, o);
        if (lane >= (u32)o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    u64 carry = 0, all = 0;
#pragma unroll
    for (int w = 0; w < EM_THREADS / 32; ++w) {
        u64 c = s_warp[w];
        if ((u32)w < warp) carry += c;
        all += c;
    }
    *total = all;
    __syncthreads();
    return carry + inc - v;
}

__global__ void __launch_bounds__(EM_THREADS) k_emit(const u64* __restrict__ rec, u64 n, Layout lay, u64* __restrict__ cand,
                                                    u64 win_lo, u64 win_hi, int first_round, u64* tile_prefix,
                                                    u64* lb_status, DevInfo* info) {
    __shared__ u64 s_rec[EM_TILE + 1];   // s_rec[0] = record before the tile
    __shared__ u64 s_scan[EM_TILE + 1];  // exclusive pair offsets inside the tile
    __shared__ i64 s_a[EM_TILE];         // partner range start (global position)
    __shared__ u64 s_warp64[EM_THREADS / 32 + 1];
    __shared__ i32 s_warp32[EM_THREADS / 32];
    __shared__ i64 s_tile_rs;
    __shared__ u64 s_excl;

    const u32 tid = threadIdx.x;
    const u32 tile = blockIdx.x;
    if (!first_round) {
        // skip tiles whose pairs lie entirely outside the window
        const u64 lo = tile_prefix[2 * tile], cnt = tile_prefix[2 * tile + 1];
        if (cnt == 0 || lo + cnt <= win_lo || lo >= win_hi) return;
    }
    const u64 base = (u64)tile * EM_TILE;
    const u32 tile_n = (u32)min((u64)EM_TILE, n - base);
    const int idb = lay.id_bits;
    const u64 idmask = (1ull << idb) - 1ull;

    for (u32 i = tid; i < tile_n; i += EM_THREADS) s_rec[i + 1] = rec[base + i];
    if (tid == 0) s_rec[0] = base > 0 ? rec[base - 1] : 0ull;
    __syncthreads();

    if (tid == 0) {
        // run start of the tile's first record when that run began in an earlier tile
        i64 rs = (i64)base;
        if (base > 0 && (s_rec[0] >> idb) == (s_rec[1] >> idb)) {
            const u64 target = (s_rec[1] >> idb) << idb;  // smallest record with this hash
            u64 lo = 0, hi = base - 1;                     // rec[hi] has the hash; find first pos with rec >= target
            while (lo < hi) {
                u64 mid = (lo + hi) >> 1;
                if (rec[mid] >= target) hi = mid; else lo = mid + 1;
            }
            rs = (i64)lo;
        }
        s_tile_rs = rs;
    }

    // ---- run starts: max-scan of head positions ----
    i32 rs_local[EM_IPT];
    i32 last = -1;
#pragma unroll
    for (int k = 0; k < EM_IPT; ++k) {
        const u32 pos = tid * EM_IPT + k;
        if (pos < tile_n) {
            const bool head = (base + pos == 0) || ((s_rec[pos] >> idb) != (s_rec[pos + 1] >> idb));
            if (head) last = (i32)pos;
        }
        rs_local[k] = last;
    }
    const i32 carry = sd_block_excl_max<EM_THREADS>(last, s_warp32);  // contains __syncthreads: s_tile_rs visible
    const i64 tile_rs = s_tile_rs;

    // ---- partner ranges and pair counts ----
    u64 pc[EM_IPT], tsum = 0;
#pragma unroll
    for (int k = 0; k < EM_IPT; ++k) {
        const u32 pos = tid * EM_IPT + k;
        pc[k] = 0;
        if (pos < tile_n) {
            const i32 r = rs_local[k] >= 0 ? rs_local[k] : carry;
            const i64 rs = r >= 0 ? (i64)base + r : tile_rs;
            const i64 gpos = (i64)base + pos;
            i64 b = gpos;
            if (lay.cross) {
                const u64 me = s_rec[pos + 1];
                if ((me & idmask) < (u64)lay.n_a) {
                    b = rs;  // query record: pairs with nothing
                } else {
                    // first position in [rs, gpos] whose id is a reference id
                    i64 lo = rs, hi = gpos;
                    while (lo < hi) {
                        i64 mid = (lo + hi) >> 1;
                        const u64 x = mid >= (i64)base - 1 ? s_rec[mid - (i64)base + 1] : rec[mid];
                        if ((x & idmask) >= (u64)lay.n_a) hi = mid; else lo = mid + 1;
                    }
                    b = lo;
                }
            }
            s_a[pos] = rs;
            pc[k] = (u64)(b - rs);
            tsum += pc[k];
        }
    }
    u64 T;
    u64 run = block_excl_sum64(tsum, &T, s_warp64);
#pragma unroll
    for (int k = 0; k < EM_IPT; ++k) {
        const u32 pos = tid * EM_IPT + k;
        if (pos < tile_n) s_scan[pos] = run;
        run += pc[k];
    }
    if (tid == 0) {
        s_scan[tile_n] = T;
        // Output slots: the ORDER of candidates is irrelevant (they are sorted next), so a tile claims
        // its range with one atomic add instead of an ordered scan across tiles; the claimed base is
        // saved so that later windows of the same call see the same numbering.
        u64 excl;
        if (first_round) {
            excl = T ? (u64)atomicAdd((unsigned long long*)&info->n_cand, (unsigned long long)T) : 0ull;
            tile_prefix[2 * tile] = excl;
            tile_prefix[2 * tile + 1] = T;
        } else {
            excl = tile_prefix[2 * tile];
        }
        s_excl = excl;
    }
    __syncthreads();
    const u64 excl = s_excl;
    if (T == 0 || excl + T <= win_lo || excl >= win_hi) return;

    // ---- write pairs by flat index ----
    const u64 p_lo = win_lo > excl ? win_lo - excl : 0ull;
    const u64 p_hi = min(T, win_hi - excl);
    for (u64 p = p_lo + tid; p < p_hi; p += EM_THREADS) {
        u32 lo = 0, hi = tile_n;  // largest idx with s_scan[idx] <= p
        while (hi - lo > 1) {
            u32 mid = (lo + hi) >> 1;
            if (s_scan[mid] <= p) lo = mid; else hi = mid;
        }
        const i64 ppos = s_a[lo] + (i64)(p - s_scan[lo]);
        const u64 partner = ppos >= (i64)base - 1 ? s_rec[ppos - (i64)base + 1] : rec[ppos];
        const u64 a_id = partner & idmask;
        u64 b_id = s_rec[lo + 1] & idmask;
        if (lay.cross) b_id -= (u64)lay.n_a;
        cand[excl + p - win_lo] = (a_id << lay.b_bits) | b_id;
    }
}

}  // namespace

i64 sd_emit_tiles(i64 n_records) { return (n_records + EM_TILE - 1) / EM_TILE; }

cudaError_t sd_emit(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 win_lo, u64 win_hi,
                    int first_round, u64* tile_prefix, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = sd_emit_tiles(n_records);
    if (tiles == 0) return cudaSuccess;
    if (first_round) {
        cudaError_t e = cudaMemsetAsync(&info->n_cand, 0, sizeof(u64), st);
        if (e != cudaSuccess) return e;
    }
    k_emit<<<(unsigned)tiles, EM_THREADS, 0, st>>>(records, (u64)n_records, lay, cand, win_lo, win_hi, first_round,
                                                    tile_prefix, lb_status, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}
