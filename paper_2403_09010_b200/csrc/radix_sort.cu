// radix_sort.cu — S2/K2: stable LSD radix sort of 64-bit records, onesweep style.
//
// "Second, sort those tuples by the deletion variant.  This guarantees that all strings with
// matching deletion variants will be stored contiguously." (§I.B step 2; App. F.2
// step 2; App. F.3 step 2).  The paper's tools use a parallel CPU sort
// and a GPU merge sort; this is a hand-written least-significant-digit radix sort instead:
//   * one up-front pass builds the 256-bin histogram of every digit place (k_histogram) — the
//     variant-generation kernel fuses this into its own pass and skips the extra read;
//   * one kernel per 8-bit digit (k_onesweep): each tile ranks its keys with warp-level match
//     groups and per-warp shared-memory counters, obtains its cross-tile exclusive prefix per digit
//     by decoupled look-back over a status array (tile order = atomic ticket, so predecessors have
//     always started), stages the tile in shared memory in digit order and writes each digit's keys
//     to one contiguous global segment.
// Every pass reads n*8 and writes n*8 bytes: the algorithmic traffic of the sort is 16 B/record/pass.
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
    __shared__ u32 s_warp[9];
    u32* h = ghist + blockIdx.x * 256;
    u32 v = h[threadIdx.x], total;
    u32 e = sd_block_excl_sum<256>(v, &total, s_warp);
    h[threadIdx.x] = e;
}

// ---------------------------------------------------------------------------------------------
#define OS_FLAG_AGG (1u << 30)
#define OS_FLAG_PRE (2u << 30)
#define OS_MASK ((1u << 30) - 1)

template <int THREADS, int IPT>
__global__ void __launch_bounds__(THREADS) k_onesweep(const u64* __restrict__ in, u64* __restrict__ out, u32 n, int shift,
                                                     const u32* __restrict__ gbase, u32* __restrict__ status,
                                                     u32* __restrict__ ticket) {
    constexpr int TILE = THREADS * IPT, NW = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* skeys = reinterpret_cast<u64*>(smem_raw);   // TILE keys, digit order
    u32* whist = reinterpret_cast<u32*>(skeys + TILE);  // NW x 256 per-warp digit counters
    u32* s_tstart = whist + NW * 256;                 // 256: start of each digit inside the tile
    u32* s_gofs = s_tstart + 256;                     // 256: global offset of digit d minus s_tstart[d]
    __shared__ u32 s_tile;
    __shared__ u32 s_warp[NW + 1];

    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < NW * 256; i += THREADS) whist[i] = 0;
    __syncthreads();
    const u32 tile = s_tile;
    const u32 base = tile * TILE;
    const u32 tile_n = min((u32)TILE, n - base);
    const u32 wbase = warp * (32 * IPT);

    // ---- load, warp-striped: item k of lane l is tile position wbase + 32k + l (coalesced) ----
    u64 key[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        u32 pos = wbase + 32 * k + lane;
        key[k] = pos < tile_n ? in[base + pos] : ~0ull;
    }

    // ---- rank inside the warp's chunk (stable: position order = (k, lane)) ----
    u32* myhist = whist + warp * 256;
    const u32 lane_lt = (1u << lane) - 1u;
    unsigned short rank[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const bool valid = (wbase + 32 * k + lane) < tile_n;
        const u32 dg = valid ? ((u32)(key[k] >> shift) & 255u) : 256u;
        const u32 peers = __match_any_sync(SD_FULL, dg);
        const u32 below = __popc(peers & lane_lt);
        u32 pre = 0;
        if (below == 0 && valid) {
            pre = myhist[dg];
            myhist[dg] = pre + __popc(peers);
        }
        pre = __shfl_sync(SD_FULL, pre, __ffs(peers) - 1);
        rank[k] = (unsigned short)(pre + below);
        __syncwarp();
    }
    __syncthreads();

    // ---- per-digit: exclusive offsets across warps, tile total, look-back ----
    u32 total = 0;
    if (tid < 256) {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            u32 c = whist[w * 256 + tid];
            whist[w * 256 + tid] = total;
            total += c;
        }
    }
    u32 tile_sum;
    u32 tstart = sd_block_excl_sum<THREADS>(total, &tile_sum, s_warp);
    if (tid < 256) {
        s_tstart[tid] = tstart;
        u32 excl = 0;
        u32* st = status + (u64)tile * 256 + tid;
        if (tile == 0) {
            sd_st_relaxed32(st, OS_FLAG_PRE | total);
        } else {
            sd_st_relaxed32(st, OS_FLAG_AGG | total);
            const u32* p = st - 256;
            while (true) {
                u32 s;
                do { s = sd_ld_relaxed32(p); } while ((s >> 30) == 0);
                excl += s & OS_MASK;
                if ((s >> 30) == 2) break;
                p -= 256;
            }
            sd_st_relaxed32(st, OS_FLAG_PRE | (excl + total));
        }
        s_gofs[tid] = gbase[tid] + excl - tstart;
    }
    __syncthreads();

    // ---- scatter into shared memory in digit order ----
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        if ((wbase + 32 * k + lane) < tile_n) {
            const u32 dg = (u32)(key[k] >> shift) & 255u;
            skeys[s_tstart[dg] + myhist[dg] + rank[k]] = key[k];
        }
    }
    __syncthreads();

    // ---- write out: consecutive threads -> consecutive slots of one digit's global segment ----
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        u32 pos = tid + k * THREADS;
        if (pos < tile_n) {
            u64 kk = skeys[pos];
            u32 dg = (u32)(kk >> shift) & 255u;
            out[s_gofs[dg] + pos] = kk;
        }
    }
}

constexpr int OS_THREADS = 256;
constexpr int OS_IPT = 16;
constexpr int OS_TILE = OS_THREADS * OS_IPT;
constexpr size_t OS_SMEM = (size_t)OS_TILE * 8 + (OS_THREADS / 32) * 256 * 4 + 2 * 256 * 4;

}  // namespace

// ---------------------------------------------------------------------------------------------
i64 sd_sort_tiles(i64 n) { return (n + OS_TILE - 1) / OS_TILE; }

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

// Runs the passes.  The histograms in `scratch` must be complete (raw counts).  Returns in *result
// the buffer (keys or tmp) that holds the sorted records.
cudaError_t sd_sort_passes(u64* keys, u64* tmp, i64 n, int begin_bit, int npass, void* scratch, cudaStream_t st,
                           u64** result, i64* launches) {
    *result = keys;
    if (n == 0 || npass == 0) return cudaSuccess;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_onesweep<OS_THREADS, OS_IPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)OS_SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    u32* hist = sd_sort_hist_ptr(scratch);
    u32* tickets = hist + npass * 256;
    u32* status = tickets + 64;
    const i64 tiles = sd_sort_tiles(n);
    k_hist_scan<<<npass, 256, 0, st>>>(hist);
    if (launches) ++*launches;
    u64 *src = keys, *dst = tmp;
    for (int p = 0; p < npass; ++p) {
        k_onesweep<OS_THREADS, OS_IPT><<<(unsigned)tiles, OS_THREADS, OS_SMEM, st>>>(
            src, dst, (u32)n, begin_bit + 8 * p, hist + p * 256, status + (size_t)p * tiles * 256, tickets + p);
        if (launches) ++*launches;
        std::swap(src, dst);
    }
    *result = src;
    return cudaGetLastError();
}
