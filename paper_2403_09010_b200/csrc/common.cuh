// common.cuh — device helpers shared by the libsymdel kernels (sm_100a).
// Nothing here is shared with oracle/ (the CPU oracle has its own, different, arithmetic).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef uint64_t u64;
typedef uint32_t u32;
typedef int64_t i64;
typedef int32_t i32;

#define SD_FULL 0xffffffffu
#define SD_L_MAX 64  // longest sequence (one Myers word) = SYMDEL_L_MAX of include/symdel.h
#define SD_D_MAX 4   // = SYMDEL_D_MAX

// ---- device status block (one per call, in the workspace; copied to pinned host memory) --------
struct DevInfo {
    u64 nmax;        // sum over sequences of V(L, d) (deletion sets)
    u64 n_records;   // records written by the last generate
    u64 n_cand;      // candidate pairs counted by the last emit
    u64 n_surv;      // survivors appended so far
    u64 n_out;       // final output pairs
    u64 n_unique;    // unique candidates seen by verify (statistics)
    u32 maxlen;      // longest sequence
    u32 err;         // bit flags, see below
    u32 ticket[8];   // dynamic tile tickets (one per kernel family)
    u64 nmax_b;      // the part of nmax that comes from set B (cross-search)
    u64 win_end;     // join: end (flat pair index) of what the last round wrote
    u32 join_fallback;  // k_join_fast: 1 = a tile's list overflowed, 2 = the pairs do not fit the window
    u32 join_redo;      // k_join_fast: tiles on the redo list (keep right after join_fallback: cleared together)
    u64 nofit_inv;      // k_join_bkt: ~(smallest claim base that did not fit the window), 0 = every claim fit (keep right after join_redo: cleared together)
    u32 part_overflow;  // fused pipeline: 1 = a level-1 bin was full, 2 = a level-2 bucket was full
    u32 surv_overflow;  // k_verify: the survivors of this flush did not fit behind the survivor list (nothing lost: the host merges the list and repeats the flush)
    u64 residues;       // sum of the (prefix-truncated) sequence lengths
    u64 n_filt;         // candidates of the current window that passed the duplicate filter (k_cand_filter)
    u32 len_hist[SD_L_MAX + 1];  // sequences per (prefix-truncated) length: the host lays the key-range chunks out over the variant lengths
};
enum { SD_ERR_OFFSETS = 1, SD_ERR_TOO_LONG = 2, SD_ERR_RESIDUE = 4, SD_ERR_INTERNAL = 8, SD_ERR_OVERFLOW = 16 };
enum { SD_TK_SORT = 0, SD_TK_EMIT = 1, SD_TK_VERIFY = 2, SD_TK_FINAL = 3, SD_TK_SCAN = 4 };

// ---- programmatic dependent launch (PDL; SASS: ACQBULK / griddepcontrol) ----------------------------------------
// The record kernels and the sort passes run back to back on one stream.  A kernel launched with sd_launch_dep may be
// scheduled while its predecessor drains; it must call sd_dep_wait() before it touches anything the predecessor wrote
// (here: as its first statement, so the semantics are those of plain stream order — what is gained is the launch latency
// and the ramp of the next grid).  sd_dep_release() lets the successor in once every block of this grid has started.
__device__ __forceinline__ void sd_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void sd_dep_release() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t sd_launch_dep(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st,
                                        Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- decoupled look-back, one 64-bit value per tile ---------------------------------------------
// status word: bits 63:62 = flag (0 invalid, 1 aggregate, 2 inclusive prefix), bits 61:0 = value.
// A tile publishes its aggregate, then walks its predecessors summing aggregates until it meets an
// inclusive prefix, then publishes its own inclusive prefix.  Tiles get their index from an atomic
// ticket, so every predecessor has started and the spin always terminates.  Flag and value share
// one word, so a single relaxed 64-bit store/load is enough (no fence between flag and payload).
#define SD_LB_AGG (1ull << 62)
#define SD_LB_PRE (2ull << 62)
#define SD_LB_MASK ((1ull << 62) - 1)

__device__ __forceinline__ u64 sd_ld_relaxed(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void sd_st_relaxed(u64* p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ u32 sd_ld_relaxed32(const u32* p) {
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void sd_st_relaxed32(u32* p, u32 v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Called by all 32 lanes of ONE converged warp; inspects 32 predecessors per
// round trip (lane 0 = nearest), so the walk back to the closest inclusive prefix costs
// ceil(depth / 32) L2 latencies instead of depth.  Returns the exclusive prefix to every lane.
__device__ __forceinline__ u64 sd_lookback_warp(u64* status, u32 tile, u64 aggregate) {
    const u32 lane = threadIdx.x & 31;
    if (tile == 0) {
        if (lane == 0) sd_st_relaxed(status, SD_LB_PRE | aggregate);
        return 0;
    }
    if (lane == 0) sd_st_relaxed(status + tile, SD_LB_AGG | aggregate);
    u64 excl = 0;
    i64 hi = (i64)tile;
    while (true) {
        const i64 idx = hi - 1 - (i64)lane;
        u64 s = SD_LB_PRE;  // virtual tile before tile 0: inclusive prefix 0
        if (idx >= 0) {
            do { s = sd_ld_relaxed(status + idx); } while ((s >> 62) == 0);
        }
        const u32 pre = __ballot_sync(SD_FULL, (s >> 62) == 2);
        u64 v = s & SD_LB_MASK;
        if (pre && lane > (u32)(__ffs(pre) - 1)) v = 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SD_FULL, v, o);
        excl += v;
        if (pre) break;
        hi -= 32;
    }
    if (lane == 0) sd_st_relaxed(status + tile, SD_LB_PRE | (excl + aggregate));
    return excl;
}

// ---- block-wide exclusive scans (THREADS a multiple of 32, <= 1024) ------------------------------
template <int THREADS>
__device__ __forceinline__ u32 sd_block_excl_sum(u32 v, u32* total, u32* s_warp /* [THREADS/32 + 1] */) {
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u32 inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(SD_FULL, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        u32 w = lane < THREADS / 32 ? s_warp[lane] : 0;
        u32 winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(SD_FULL, winc, o);
            if (lane >= o) winc += t;
        }
        if (lane < THREADS / 32) s_warp[lane] = winc - w;
        if (lane == 31) s_warp[THREADS / 32] = winc;
    }
    __syncthreads();
    u32 r = s_warp[warp] + inc - v;
    *total = s_warp[THREADS / 32];
    __syncthreads();  // s_warp may be reused by the caller
    return r;
}
