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
// Runs are short on this workload (a run of m records holds m distinct sequences sharing one variant),
// so each record finds its partners by walking BACKWARDS from its own position while the hash matches
// (plain global loads: they hit L1/L2, the tile was just streamed in); the walk costs what the pairs it
// emits cost.  The kernel keeps no tile in shared memory: one coalesced 8-byte load per record, the
// left neighbour by warp shuffle.  Counts are scanned inside the block, the tile claims its output range with ONE atomic
// add (candidate order is irrelevant: they are sorted next) and every record then writes its own
// pairs.  Only pairs whose flat index lies in [win_lo, win_hi) are written: when the candidate buffer
// is smaller than the total, the host replays the kernel once per window (later rounds reuse the
// saved per-tile base and count, so the numbering is the same in every round of one call).
#include "kernels.h"

namespace {

constexpr int EM_THREADS = 256, EM_IPT = 16, EM_TILE = EM_THREADS * EM_IPT;

__global__ void __launch_bounds__(EM_THREADS) k_emit(const u64* __restrict__ rec, u64 n, Layout lay, u64* __restrict__ cand,
                                                    u64 win_lo, u64 win_hi, int first_round, u64* tile_prefix,
                                                    DevInfo* info) {
    __shared__ u64 s_wsum[EM_THREADS / 32];
    __shared__ u64 s_excl;

    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 tile = blockIdx.x;
    if (!first_round) {
        const u64 lo = tile_prefix[2 * tile], cnt = tile_prefix[2 * tile + 1];
        if (cnt == 0 || lo + cnt <= win_lo || lo >= win_hi) return;  // nothing of this tile in the window
    }
    const i64 base = (i64)tile * EM_TILE;
    const u32 tile_n = (u32)min((u64)EM_TILE, n - (u64)base);
    const int idb = lay.id_bits;
    const u64 idmask = (1ull << idb) - 1ull;
    const u64 n_a = (u64)lay.n_a;
    const bool cross = lay.cross != 0;

    // ---- phase 1: every record and its left neighbour straight from global memory (coalesced; the
    //      neighbour comes from the lane below).  `cont` marks the few records that continue a run;
    //      only those walk back, in a compact loop (keeps the unrolled part tiny). ----
    const u64 hlim = 1ull << idb;  // same hash <=> (x ^ y) < 2^id_bits
    u32 cont = 0;
#pragma unroll
    for (int k = 0; k < EM_IPT; ++k) {
        const u32 pos = k * EM_THREADS + tid;
        const u64 me = pos < tile_n ? rec[base + pos] : ~0ull;
        u64 prev = __shfl_up_sync(SD_FULL, me, 1);
        if (lane == 0) prev = (pos < tile_n && base + pos > 0) ? rec[base + pos - 1] : ~me;
        const bool same = pos < tile_n && ((me ^ prev) < hlim) && (!cross || (me & idmask) >= n_a);
        cont |= (same ? 1u : 0u) << k;
    }
    u64 tsum = 0;
    for (u32 m = cont; m; m &= m - 1) {
        const i64 g = base + (i64)((__ffs(m) - 1) * EM_THREADS + tid);
        const u64 me = rec[g];
        i64 gp = g - 1;
        while (gp >= 0) {
            const u64 x = rec[gp];
            if ((x ^ me) >= hlim) break;
            tsum += (!cross || (x & idmask) < n_a) ? 1u : 0u;  // cross: partners are the run's queries
            --gp;
        }
    }
    // ---- block exclusive scan of the per-thread totals ----
    u64 inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u64 t = __shfl_up_sync(SD_FULL, inc, o);
        if (lane >= (u32)o) inc += t;
    }
    if (lane == 31) s_wsum[warp] = inc;
    __syncthreads();
    u64 carry = 0, T = 0;
#pragma unroll
    for (int w = 0; w < EM_THREADS / 32; ++w) {
        const u64 c = s_wsum[w];
        if ((u32)w < warp) carry += c;
        T += c;
    }
    if (T == 0) {
        if (first_round && tid == 0) tile_prefix[2 * tile] = 0, tile_prefix[2 * tile + 1] = 0;
        return;
    }
    if (tid == 0) {
        u64 excl;
        if (first_round) {
            excl = (u64)atomicAdd((unsigned long long*)&info->n_cand, (unsigned long long)T);
            tile_prefix[2 * tile] = excl;
            tile_prefix[2 * tile + 1] = T;
        } else {
            excl = tile_prefix[2 * tile];
        }
        s_excl = excl;
    }
    __syncthreads();
    u64 flat = s_excl + carry + inc - tsum;  // flat index of this thread's first pair
    if (tsum == 0 || flat + tsum <= win_lo || flat >= win_hi) return;

    // ---- phase 2: every run-continuing record writes its own pairs (same walk) ----
    for (u32 m = cont; m; m &= m - 1) {
        const i64 g = base + (i64)((__ffs(m) - 1) * EM_THREADS + tid);
        const u64 me = rec[g];
        const u64 b_id = cross ? (me & idmask) - n_a : (me & idmask);
        i64 gp = g - 1;
        while (gp >= 0) {
            const u64 x = rec[gp];
            if ((x ^ me) >= hlim) break;
            --gp;
            if (cross && (x & idmask) >= n_a) continue;  // a reference record of the same run
            if (flat >= win_lo && flat < win_hi) cand[flat - win_lo] = ((x & idmask) << lay.b_bits) | b_id;
            ++flat;
        }
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
    (void)lb_status;
    k_emit<<<(unsigned)tiles, EM_THREADS, 0, st>>>(records, (u64)n_records, lay, cand, win_lo, win_hi, first_round,
                                                    tile_prefix, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}
