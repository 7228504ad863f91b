// verify.cu — S3b (unique) + S4/K6 (verification) + result unpacking.
//
// "Deduplicate {(i, i')}.  Calculate the sequences' distance, filter for threshold validity, then
// return {(i, i', d(s_i, s_i'))}" (App. F.1 steps 4-5; App. F.3 steps 4-5,
// PAPER.md:350-351).  Duplicates and false positives of the lookup "can be filtered with
// post-processing verification"; verification is on the FULL sequences, so the
// hash used as the join key cannot change the result.
//
// The candidates arrive sorted (radix sort of the packed pair ids), so "unique" is a comparison with
// the left neighbour, fused into the verifier.  The distance is the bit-parallel global edit
// distance of Myers (1999) in Hyyro's (2003) formulation: one machine word holds a column of
// vertical deltas of the Wagner-Fischer table (pattern length <= 64, or <= 32 on the 32-bit path);
// per text character it costs ~15 bit operations instead of a column of min/add.  The match mask
// Eq[c] is rebuilt from five bit-planes of the pattern's 5-bit residue codes (3 logic ops per plane
// pair) rather than looked up in a 32-entry table, which keeps the whole state in registers.
// Survivors are compacted in order (block scan + decoupled look-back), so the output stays sorted.
#include "kernels.h"

namespace {

template <typename W>
__device__ __forceinline__ int myers_lev(const int8_t* __restrict__ p, int m, const int8_t* __restrict__ t, int n) {
    if (m == 0) return n;
    if (n == 0) return m;
    W b0 = 0, b1 = 0, b2 = 0, b3 = 0, b4 = 0;
    for (int j = 0; j < m; ++j) {
        const W c = (W)(unsigned char)p[j];
        b0 |= (c & 1) << j;
        b1 |= ((c >> 1) & 1) << j;
        b2 |= ((c >> 2) & 1) << j;
        b3 |= ((c >> 3) & 1) << j;
        b4 |= ((c >> 4) & 1) << j;
    }
    const W mask = (m == (int)(8 * sizeof(W))) ? ~(W)0 : (((W)1 << m) - 1);
    const W top = (W)1 << (m - 1);
    W Pv = mask, Mv = 0;
    int score = m;
    for (int i = 0; i < n; ++i) {
        const unsigned c = (unsigned char)t[i];
        W Eq = mask;
        Eq &= (c & 1) ? b0 : ~b0;
        Eq &= (c & 2) ? b1 : ~b1;
        Eq &= (c & 4) ? b2 : ~b2;
        Eq &= (c & 8) ? b3 : ~b3;
        Eq &= (c & 16) ? b4 : ~b4;
        const W Xv = Eq | Mv;
        const W Xh = (((Eq & Pv) + Pv) ^ Pv) | Eq;
        W Ph = Mv | ~(Xh | Pv);
        W Mh = Pv & Xh;
        score += (Ph & top) ? 1 : 0;
        score -= (Mh & top) ? 1 : 0;
        Ph = (Ph << 1) | 1;  // first-row boundary D[0][j] = j: global (whole-string) distance
        Mh = Mh << 1;
        Pv = (Mh | ~(Xv | Ph)) & mask;
        Mv = Ph & Xv & mask;
    }
    return score;
}

__device__ __forceinline__ int lev_dispatch(const int8_t* p, int m, const int8_t* t, int n, bool narrow) {
    // the shorter string is the pattern (fewer word bits; the distance is symmetric)
    if (m > n) {
        const int8_t* x = p; p = t; t = x;
        int y = m; m = n; n = y;
    }
    return narrow ? myers_lev<u32>(p, m, t, n) : myers_lev<u64>(p, m, t, n);
}

constexpr int VF_THREADS = 256;

__global__ void __launch_bounds__(VF_THREADS) k_verify(const u64* __restrict__ cand, u64 n, SeqSetDev A, SeqSetDev B,
                                                      Layout lay, int narrow, u64* __restrict__ surv, u64 surv_base,
                                                      u64 surv_capacity, u64* lb_status, DevInfo* info) {
    __shared__ u32 s_warp[VF_THREADS / 32 + 1];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl;
    const u32 tid = threadIdx.x;
    if (tid == 0) {
        s_tile = atomicAdd(&info->ticket[SD_TK_VERIFY], 1u);
        if (s_tile == gridDim.x - 1) info->ticket[SD_TK_VERIFY] = 0;
    }
    __syncthreads();
    const u32 tile = s_tile;
    const u64 t = (u64)tile * VF_THREADS + tid;
    bool uniq = false, keep = false;
    u64 c = 0;
    int dist = 0;
    if (t < n) {
        c = cand[t];
        uniq = (t == 0) || (cand[t - 1] != c);
        const u64 a = c >> lay.b_bits, b = c & ((1ull << lay.b_bits) - 1ull);
        if (!lay.cross && a == b) uniq = false;  // same sequence twice in one run (hash collision / no thinning)
        if (uniq) {
            const i64 pa = A.off[a], pb = B.off[b];
            const int la = (int)(A.off[a + 1] - pa), lb = (int)(B.off[b + 1] - pb);
            const int dl = la > lb ? la - lb : lb - la;
            if (dl <= lay.d) {
                dist = lev_dispatch(A.seqs + pa, la, B.seqs + pb, lb, narrow != 0);
                keep = dist <= lay.d;
            }
        }
    }
    u32 total;
    const u32 rank = sd_block_excl_sum<VF_THREADS>(keep ? 1u : 0u, &total, s_warp);
    const u32 nuniq = __syncthreads_count(uniq);
    if (tid < 32) {
        const u64 excl = sd_lookback_warp(lb_status, tile, total);
        if (tid == 0) {
            s_excl = excl;
            if (nuniq) atomicAdd((unsigned long long*)&info->n_unique, (unsigned long long)nuniq);
            if (tile == gridDim.x - 1) info->n_surv = surv_base + excl + total;
        }
    }
    __syncthreads();
    if (keep) {
        const u64 pos = surv_base + s_excl + rank;
        if (pos < surv_capacity) surv[pos] = (c << 3) | (u64)dist;
        else atomicOr(&info->err, (u32)SD_ERR_OVERFLOW);
    }
}

constexpr int FN_THREADS = 256;

__global__ void __launch_bounds__(FN_THREADS) k_finalize(const u64* __restrict__ surv, u64 n, Layout lay, int dedup,
                                                        i32* __restrict__ out_i, i32* __restrict__ out_j,
                                                        i32* __restrict__ out_dist, u64 capacity, u64* lb_status,
                                                        DevInfo* info) {
    __shared__ u32 s_warp[FN_THREADS / 32 + 1];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl;
    const u32 tid = threadIdx.x;
    if (tid == 0) {
        s_tile = atomicAdd(&info->ticket[SD_TK_FINAL], 1u);
        if (s_tile == gridDim.x - 1) info->ticket[SD_TK_FINAL] = 0;
    }
    __syncthreads();
    const u32 tile = s_tile;
    const u64 t = (u64)tile * FN_THREADS + tid;
    bool keep = false;
    u64 v = 0;
    if (t < n) {
        v = surv[t];
        keep = !dedup || t == 0 || (surv[t - 1] >> 3) != (v >> 3);
    }
    u32 total;
    const u32 rank = sd_block_excl_sum<FN_THREADS>(keep ? 1u : 0u, &total, s_warp);
    if (tid < 32) {
        const u64 excl = sd_lookback_warp(lb_status, tile, total);
        if (tid == 0) {
            s_excl = excl;
            if (tile == gridDim.x - 1) info->n_out = excl + total;
        }
    }
    __syncthreads();
    if (keep) {
        const u64 pos = s_excl + rank;
        if (pos < capacity) {
            const u64 pr = v >> 3;
            out_i[pos] = (i32)(pr >> lay.b_bits);
            out_j[pos] = (i32)(pr & ((1ull << lay.b_bits) - 1ull));
            out_dist[pos] = (i32)(v & 7ull);
        }
    }
}

__global__ void __launch_bounds__(256) k_lev_pairs(SeqSetDev A, SeqSetDev B, const i32* __restrict__ ia,
                                                   const i32* __restrict__ ib, i64 n, i32* __restrict__ dist) {
    const i64 t = (i64)blockIdx.x * 256 + threadIdx.x;
    if (t >= n) return;
    const i64 a = ia[t], b = ib[t];
    const i64 pa = A.off[a], pb = B.off[b];
    const int la = (int)(A.off[a + 1] - pa), lb = (int)(B.off[b + 1] - pb);
    const bool narrow = (t & 1) && la <= 32 && lb <= 32;  // exercise both word widths
    dist[t] = lev_dispatch(A.seqs + pa, la, B.seqs + pb, lb, narrow);
}

}  // namespace

i64 sd_verify_tiles(i64 n) { return (n + VF_THREADS - 1) / VF_THREADS; }

cudaError_t sd_verify(const u64* cand, i64 n_cand, SeqSetDev a, SeqSetDev b, const Layout& lay, int maxlen, u64* surv,
                      u64 surv_base, u64 surv_capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = sd_verify_tiles(n_cand);
    if (tiles == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    k_verify<<<(unsigned)tiles, VF_THREADS, 0, st>>>(cand, (u64)n_cand, a, lay.cross ? b : a, lay, maxlen <= 32 ? 1 : 0, surv,
                                                     surv_base, surv_capacity, lb_status, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_finalize(const u64* surv, i64 n_surv, const Layout& lay, int dedup, i32* out_i, i32* out_j, i32* out_dist,
                        i64 capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = (n_surv + FN_THREADS - 1) / FN_THREADS;
    if (tiles == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    k_finalize<<<(unsigned)tiles, FN_THREADS, 0, st>>>(surv, (u64)n_surv, lay, dedup, out_i, out_j, out_dist, (u64)capacity,
                                                       lb_status, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_lev_pairs(SeqSetDev a, SeqSetDev b, const i32* ia, const i32* ib, i64 n_pairs, i32* dist,
                         cudaStream_t st) {
    if (n_pairs == 0) return cudaSuccess;
    k_lev_pairs<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>(a, b, ia, ib, n_pairs, dist);
    return cudaGetLastError();
}
