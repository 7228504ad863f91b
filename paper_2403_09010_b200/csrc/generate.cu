// generate.cu — S0 (input validation, record counting, offsets) and S1/K1 (variant generation).
//
// "First, generate an array containing all tuples of deletion variants and original strings for
// both the query and reference sets." (§I.B step 1; App. F.1 step 1, PAPER.md:327;
// App. F.3 step 1).  A sequence of length L has sum_{k<=d} C(L, k) deletion sets
// (reading A-1: the 0-deletion original is included).  As in SymScan, the tuple holds
// a hash of the variant and the index of the sequence, (h_ij, i) (footnote 1):
//     record = (top hash_bits of H(variant)) << id_bits | id
// H is a polynomial hash over 5-bit residue codes, H(v) = sum_k R[v_k] * B^k + (len + 1) * K mod 2^64
// (R[c], B, K: fixed odd 64-bit constants; no finaliser — the partition digits are the TOP bits of the
// polynomial itself, which the odd multipliers already mix).  With the prefix sums A[j] = sum_{t<j} R[s_t] * B^t of the SOURCE sequence, the hash of
// the variant that deletes positions p_1 < ... < p_k is
//     sum_{m=0..k} B^{-m} * (A[p_{m+1}] - A[p_m + 1]),   p_0 = -1, p_{k+1} = L,
// so a variant costs k+1 multiply-adds instead of a pass over its residues.
//
// Thinning (reading A-2; SymScan "sort ... and deduplicate"): a deletion set is kept
// only if it is the LEFTMOST embedding of its variant, i.e. no deleted position p has
// s[p] == s[q] with q the next kept position after p.  Exactly one set per distinct (variant, id)
// survives, so repeated residues produce no duplicate records.
//
// Order: the exact pipeline (k_gen2 / k_generate) writes records in ascending id, at rec_off[id] + rank,
// where rec_off is the exclusive scan of the per-sequence counts produced by the count pass — no atomics,
// deterministic layout.  The fused pipeline (k_gen2_part / k_generate_part, the default) skips counting:
// records are staged under their top 8 hash bits and flushed to fixed-capacity bins in arbitrary order.
#include <cstddef>

#include "kernels.h"

namespace {

__constant__ u64 c_R[32];
__constant__ u64 c_Bpow[SD_L_MAX + 1];
__constant__ u64 c_Binv[SD_D_MAX + 1];
__constant__ u32 c_binom[(SD_L_MAX + 1) * (SD_D_MAX + 1)];  // C(n, k)
__constant__ u32 c_vcum[(SD_L_MAX + 1) * (SD_D_MAX + 2)];   // sum_{j<k} C(n, j)

constexpr u64 K_LEN = 0x9fb21c651e98df25ull;

// Key-range chunks (S5).  Variants of different LENGTHS never meet, so the chunks are laid out along the axis
// (variant length, hash fraction): position = vlen << 32 | f(low word of the hash), chunk = [chunk_lo, chunk_hi).  A
// sequence of length L only has to enumerate the deletion depths k whose variant length L - k reaches into the chunk —
// over all chunks every deletion set is enumerated once, except at the lengths a chunk boundary cuts (those are split
// by the hash fraction: a function of the LOW word only, so the partitioned top bits stay uniform inside every chunk).
__device__ __forceinline__ bool gen_in_chunk(u64 h, u32 vlen, u64 lo, u64 hi) {
    const u64 pos = ((u64)vlen << 32) | (u64)((u32)h * 0x9e3779b1u);
    return pos >= lo && pos < hi;
}
// does any record of variant length vlen belong to the chunk?
__device__ __forceinline__ bool gen_len_in_chunk(u32 vlen, u64 lo, u64 hi) { return (((u64)vlen + 1) << 32) > lo && ((u64)vlen << 32) < hi; }

// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_prepare(SeqSetDev s, int d, int is_b, int prefix, DevInfo* info) {
    // V(L, d) for every length, in shared memory: the lanes of a warp ask for different lengths, which the constant
    // cache would serve one address at a time
    __shared__ u32 s_v[SD_L_MAX + 1];
    __shared__ u64 s_nmax[8], s_res[8];
    __shared__ u32 s_maxlen[8], s_err[8];
    __shared__ u32 s_lh[SD_L_MAX + 1];  // sequences of this block per (truncated) length
    if (threadIdx.x <= SD_L_MAX) s_v[threadIdx.x] = c_vcum[threadIdx.x * (SD_D_MAX + 2) + d + 1], s_lh[threadIdx.x] = 0;
    __syncthreads();
    u64 nmax = 0, res = 0;
    u32 maxlen = 0, err = 0;
    const i64 stride = (i64)gridDim.x * blockDim.x;
    const i64 t0 = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    i64 a = t0 < s.n ? s.off[t0] : 0;
    for (i64 i = t0; i < s.n; i += stride) {
        const i64 b = s.off[i + 1];
        const i64 an = i + stride < s.n ? s.off[i + stride] : 0;  // (next iteration's first offset, in flight with this one's second)
        if (i == 0 && a != 0) err |= SD_ERR_OFFSETS;
        i64 L = b - a;
        if (L < 0 || a < 0) err |= SD_ERR_OFFSETS;
        else if (L > SD_L_MAX) err |= SD_ERR_TOO_LONG;
        else {
            nmax += s_v[min(L, (i64)prefix)];
            res += (u64)min(L, (i64)prefix);
            maxlen = max(maxlen, (u32)L);
            atomicAdd(&s_lh[min(L, (i64)prefix)], 1u);
        }
        a = an;
    }
    // (the residue codes are range-checked by k_pack / k_check_residues, which run only after the offsets
    //  have been found valid: a malformed offsets array must never steer a read of `seqs`)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nmax += __shfl_xor_sync(SD_FULL, nmax, o);
        res += __shfl_xor_sync(SD_FULL, res, o);
        maxlen = max(maxlen, __shfl_xor_sync(SD_FULL, maxlen, o));
        err |= __shfl_xor_sync(SD_FULL, err, o);
    }
    // one set of global atomics per BLOCK (they all hit the same few words of info)
    const u32 warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) s_nmax[warp] = nmax, s_res[warp] = res, s_maxlen[warp] = maxlen, s_err[warp] = err;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) nmax += s_nmax[w], res += s_res[w], maxlen = max(maxlen, s_maxlen[w]), err |= s_err[w];
        if (nmax) atomicAdd((unsigned long long*)&info->nmax, (unsigned long long)nmax);
        if (res) atomicAdd((unsigned long long*)&info->residues, (unsigned long long)res);
        if (nmax && is_b) atomicAdd((unsigned long long*)&info->nmax_b, (unsigned long long)nmax);
        if (maxlen) atomicMax(&info->maxlen, maxlen);
        if (err) atomicOr(&info->err, err);
    }
    if (threadIdx.x <= SD_L_MAX && s_lh[threadIdx.x]) atomicAdd(&info->len_hist[threadIdx.x], s_lh[threadIdx.x]);
}

// Residue range check on its own (the stage entry point that does not pack).  Launched after k_prepare: does
// nothing unless the offsets were valid, and then offsets[n] <= 64 n bounds the scan.
__global__ void __launch_bounds__(256) k_check_residues(SeqSetDev s, DevInfo* info) {
    if (info->err) return;
    const i64 total = s.n > 0 ? s.off[s.n] : 0;
    u32 bad = 0;
    for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (i64)gridDim.x * blockDim.x) {
        const int c = s.seqs[t];
        if (c < 1 || c > 31) bad = 1;
    }
    if (__any_sync(SD_FULL, bad) && (threadIdx.x & 31) == 0) atomicOr(&info->err, (u32)SD_ERR_RESIDUE);
}

// ---------------------------------------------------------------------------------------------
// exclusive scan of u32 counts into u64 offsets, single pass, decoupled look-back
constexpr int SC_THREADS = 256, SC_IPT = 8, SC_TILE = SC_THREADS * SC_IPT;

__global__ void __launch_bounds__(SC_THREADS) k_scan_counts(const u32* __restrict__ cnt, i64 n, u64* __restrict__ rec_off,
                                                           u64* lb_status, DevInfo* info) {
    __shared__ u32 s_warp[SC_THREADS / 32 + 1];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl;
    const u32 tid = threadIdx.x;
    if (tid == 0) {
        s_tile = atomicAdd(&info->ticket[SD_TK_SCAN], 1u);
        if (s_tile == gridDim.x - 1) info->ticket[SD_TK_SCAN] = 0;  // every ticket has been taken
    }
    __syncthreads();
    const u32 tile = s_tile;
    const i64 base = (i64)tile * SC_TILE + (i64)tid * SC_IPT;
    u32 v[SC_IPT], sum = 0;
#pragma unroll
    for (int k = 0; k < SC_IPT; ++k) {
        v[k] = (base + k) < n ? cnt[base + k] : 0;
        sum += v[k];
    }
    u32 total;
    u32 excl = sd_block_excl_sum<SC_THREADS>(sum, &total, s_warp);
    if (tid < 32) {
        const u64 e = sd_lookback_warp(lb_status, tile, total);
        if (tid == 0) s_excl = e;
    }
    __syncthreads();
    u64 run = s_excl + excl;
#pragma unroll
    for (int k = 0; k < SC_IPT; ++k) {
        if ((base + k) < n) rec_off[base + k] = run;
        run += v[k];
    }
    if (tile == gridDim.x - 1 && tid == SC_THREADS - 1) {
        rec_off[n] = s_excl + total;
        info->n_records = s_excl + total;
    }
}

// ---------------------------------------------------------------------------------------------
// General path (any d <= 4, any length <= 64).
//
// Count pass without chunking: k_count_dp, one thread per sequence, the classic distinct-subsequence
// recurrence restricted to the band of <= d deletions (h[i][j] = number of distinct strings obtained
// from the prefix of length i by deleting exactly j residues):
//     h[i][j] = h[i-1][j] + h[i-1][j-1] - h[l-1][j-(i-l)],   l = nearest earlier position of s_i
// (the subtracted term only exists when i - l <= j).  The sum over j <= d equals the number of
// leftmost-embedding deletion sets, i.e. the records k_generate writes (checked at run time).
//
// Generation: a block takes 32 sequences; the deletion sets of the group are numbered consecutively
// (sequence, then size k, then colexicographic rank) and every thread walks GEN_R CONSECUTIVE numbers:
// one unranking per thread and round, then the colex successor.  Per set: the leftmost-embedding rule
// from the per-sequence masks NE_j (bit t: s[t] != s[t+j] or t+j beyond the end), and the hash
//     H = C_k + U[p_1] + Binv*U[p_2] + Binv^2*U[p_3] + Binv^3*U[p_4]
// from the per-sequence table U[p] = A[p] - Binv*A[p+1] (same function as the fast path).  A round is
// two sweeps over the same sets: count the survivors (no hash unless chunked), block scan, then hash
// and write at the scanned offsets — no register arrays, no unrolled decode.
constexpr int GEN_THREADS = 256, GEN_G = 32, GEN_R = 8, GEN_NW = GEN_THREADS / 32;
constexpr int SEQ_STRIDE = SD_L_MAX + 4;

struct GenParams {
    SeqSetDev a, b;
    i64 groups_a, groups_total;
    i64 n_a;
    int d, width, thinning, hash_bits, id_bits, npass, hshift;  // hshift: bit of the KEY where the first counted digit starts
    u32 n_chunks, chunk;
    u64 chunk_lo, chunk_hi;
    u32 prefix;  // variants are generated from the first `prefix` residues only (App. B); >= SD_L_MAX: whole sequences
    const u64* rec_off;
    u64* records;
    u32* cnt;
    u32* ghist;
    DevInfo* info;
};

__global__ void __launch_bounds__(128) k_count_dp(SeqSetDev A, SeqSetDev B, int d, int thinning, int prefix, u32* __restrict__ cnt) {
    const i64 g = (i64)blockIdx.x * 128 + threadIdx.x;
    if (g >= A.n + B.n) return;
    const SeqSetDev& S = g < A.n ? A : B;
    const i64 i0 = g < A.n ? g : g - A.n;
    const i64 o = S.off[i0];
    const int L = min((int)(S.off[i0 + 1] - o), prefix);
    if (!thinning) {
        cnt[g] = c_vcum[L * (SD_D_MAX + 2) + d + 1];
        return;
    }
    // ring of the last d + 2 rows of h (row i lives in slot i % RING)
    constexpr int RING = SD_D_MAX + 2, W = SD_D_MAX + 1;
    u32 h[RING][W];
#pragma unroll
    for (int r = 0; r < RING; ++r)
#pragma unroll
        for (int j = 0; j < W; ++j) h[r][j] = 0;
    h[0][0] = 1;
    for (int i = 1; i <= L; ++i) {
        const int c = S.seqs[o + i - 1];
        int back = 0;  // i - l for the nearest earlier equal residue within d positions, 0 = none
        for (int t = 1; t <= d && t < i; ++t)
            if (S.seqs[o + i - 1 - t] == c) {
                back = t;
                break;
            }
        const int cur = i % RING, prv = (i - 1) % RING;
        const int dup = back ? (i - back - 1) % RING : 0;  // row l - 1 = i - back - 1
        for (int j = 0; j <= d; ++j) {
            u32 v = h[prv][j] + (j > 0 ? h[prv][j - 1] : 0u);
            if (back && j >= back) v -= h[dup][j - back];
            h[cur][j] = j <= i ? v : 0u;
        }
    }
    u32 total = 0;
    for (int j = 0; j <= d; ++j) total += h[L % RING][j];
    cnt[g] = total;
}

// LW = residues per row of U: SD_L_MAX in general, 32 when the longest (truncated) sequence fits (half the shared memory)
template <int LW>
struct GenSharedT {
    u64 U[GEN_G][LW];                // U[p] = A[p] - Binv * A[p + 1]
    u64 C[GEN_G][SD_D_MAX + 1];      // C[k] = Binv^k * A[L] + (L - k + 1) * K_LEN
    u64 NE[GEN_G][SD_D_MAX];         // NE[j-1] bit t: t + j >= L or s[t] != s[t + j]
    u64 R[32];
    u64 Bpow[SD_L_MAX + 1];
    i64 off[GEN_G];
    u32 binom[(SD_L_MAX + 1) * (SD_D_MAX + 1)];
    u32 vcum[(SD_L_MAX + 1) * (SD_D_MAX + 2)];
    u32 vbase[GEN_G + 1];
    u32 len[GEN_G];
    u32 cnt[GEN_G];
    u32 wtot[GEN_NW];
    u32 running;
    unsigned char seq[GEN_G][SEQ_STRIDE];
};
typedef GenSharedT<SD_L_MAX> GenShared;

// Walks the deletion sets numbered [f, fend) of the group and calls fn(g, L, k, p) for each.
template <typename SH, typename Fn>
__device__ __forceinline__ void gen_walk(const SH& sh, u32 f, u32 fend, u32 ng, int d, Fn&& fn) {
    int p[4] = {0, 0, 0, 0};
    u32 g = 0, L = 0, left = 0;  // left = sets remaining in the current (sequence, k) class
    int k = 0;
    while (f < fend) {
        if (left == 0) {
            u32 lo = 0, hi = ng;  // largest g with vbase[g] <= f
            while (hi - lo > 1) {
                const u32 mid = (lo + hi) >> 1;
                if (sh.vbase[mid] <= f) lo = mid; else hi = mid;
            }
            g = lo;
            L = sh.len[g];
            const u32 rr = f - sh.vbase[g];
            const u32* vc = sh.vcum + L * (SD_D_MAX + 2);
            k = 0;
            while (k < d && rr >= vc[k + 1]) ++k;
            u32 idx = rr - vc[k];
            left = sh.binom[L * (SD_D_MAX + 1) + k] - idx;
            int c = (int)L - 1;  // colexicographic unranking
#pragma unroll
            for (int j = 4; j >= 1; --j) {
                if (j <= k) {
                    if (j == 1) c = (int)idx;
                    else
                        while (sh.binom[c * (SD_D_MAX + 1) + j] > idx) --c;
                    p[j - 1] = c;
                    idx -= sh.binom[c * (SD_D_MAX + 1) + j];
                    c -= 1;
                }
            }
        }
        fn(g, L, k, p);
        // colex successor: bump the first element that can move, reset the ones below it
        bool done = false;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (!done && i < k) {
                if (i == k - 1 || p[i] + 1 < p[i + 1 < 4 ? i + 1 : 3]) {
                    ++p[i];
                    done = true;
                } else {
                    p[i] = i;
                }
            }
        }
        ++f;
        --left;
    }
}

// Leftmost-embedding rule on bit masks: D = the deleted positions; a deleted position p whose deleted run
// p, p+1, .. has length exactly j meets its next KEPT position at p + j, and must satisfy NE[j-1] bit p
// (s[p] != s[p + j], or p + j beyond the end).  k <= 4, so runs are at most 4 long.  Branch-free.
template <typename SH>
__device__ __forceinline__ bool gen_canonical(const SH& sh, u32 g, int k, const int* p) {
    u64 D = 0;
#pragma unroll
    for (int m = 0; m < 4; ++m)
        if (m < k) D |= 1ull << p[m];
    const u64 r2 = D & (D >> 1), r3 = r2 & (D >> 2), r4 = r3 & (D >> 3);
    const u64 bad = ((D & ~r2) & ~sh.NE[g][0]) | ((r2 & ~r3) & ~sh.NE[g][1]) | ((r3 & ~r4) & ~sh.NE[g][2]) | (r4 & ~sh.NE[g][3]);
    return bad == 0;
}

template <typename SH>
__device__ __forceinline__ u64 gen_hash(const SH& sh, u32 g, int k, const int* p) {
    u64 h = sh.C[g][k];
    if (k > 0) h += sh.U[g][p[0]];
    if (k > 1) h += c_Binv[1] * sh.U[g][p[1]];
    if (k > 2) h += c_Binv[2] * sh.U[g][p[2]];
    if (k > 3) h += c_Binv[3] * sh.U[g][p[3]];
    return h;
}

template <bool COUNT_ONLY, bool CHUNKED>
__global__ void __launch_bounds__(GEN_THREADS) k_generate(GenParams P) {
    extern __shared__ __align__(16) unsigned char gen_smem[];
    GenShared& sh = *reinterpret_cast<GenShared*>(gen_smem);
    u32* s_hist = reinterpret_cast<u32*>(gen_smem + sizeof(GenShared));  // [npass][256], generation only

    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < (SD_L_MAX + 1) * (SD_D_MAX + 1); i += GEN_THREADS) sh.binom[i] = c_binom[i];
    for (int i = tid; i < (SD_L_MAX + 1) * (SD_D_MAX + 2); i += GEN_THREADS) sh.vcum[i] = c_vcum[i];
    if (tid < 32) sh.R[tid] = c_R[tid];
    if (tid <= SD_L_MAX) sh.Bpow[tid] = c_Bpow[tid];
    if (!COUNT_ONLY)
        for (int i = tid; i < P.npass * 256; i += GEN_THREADS) s_hist[i] = 0;
    const int d = P.d;
    const bool thinning = P.thinning != 0;
    const int kshift = 64 - P.hash_bits;

    for (i64 gi = blockIdx.x; gi < P.groups_total; gi += gridDim.x) {
        const bool in_b = gi >= P.groups_a;
        const SeqSetDev& S = in_b ? P.b : P.a;
        const i64 first = (in_b ? gi - P.groups_a : gi) * GEN_G;
        const u32 ng = (u32)min((i64)GEN_G, S.n - first);
        const u64 gid0 = (u64)first + (in_b ? (u64)P.n_a : 0ull);
        __syncthreads();  // previous group fully consumed (also orders the table fill above)
        if (tid < GEN_G) {
            u32 L = 0;
            if (tid < ng) {
                const i64 a = S.off[first + tid];
                L = min((u32)(S.off[first + tid + 1] - a), P.prefix);
                sh.off[tid] = a;
            }
            sh.len[tid] = L;
            sh.cnt[tid] = 0;
            u32 v = tid < ng ? sh.vcum[L * (SD_D_MAX + 2) + d + 1] : 0, inc = v;  // V(L, d), scanned over the group
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u32 t = __shfl_up_sync(SD_FULL, inc, o);
                if (lane >= (u32)o) inc += t;
            }
            sh.vbase[tid + 1] = inc;
            if (tid == 0) {
                sh.vbase[0] = 0;
                sh.running = 0;
            }
        }
        __syncthreads();
        for (u32 idx = tid; idx < ng * (u32)P.width; idx += GEN_THREADS) {
            const u32 g = idx / (u32)P.width, q = idx - g * (u32)P.width;
            sh.seq[g][q] = q < sh.len[g] ? (unsigned char)S.seqs[sh.off[g] + q] : (unsigned char)0;
        }
        __syncthreads();
        if (tid < ng) {  // per-sequence tables
            const u32 L = sh.len[tid];
            const unsigned char* sq = sh.seq[tid];
            u64 acc = 0;
            for (u32 q = 0; q < L; ++q) {
                const u64 nxt = acc + sh.R[sq[q] & 31] * sh.Bpow[q];
                sh.U[tid][q] = acc - c_Binv[1] * nxt;
                acc = nxt;
            }
            for (int k = 0; k <= SD_D_MAX; ++k) sh.C[tid][k] = c_Binv[k] * acc + (u64)(L - k + 1) * K_LEN;
            for (int j = 1; j <= SD_D_MAX; ++j) {
                u64 m = 0;
                for (u32 q = 0; q < L; ++q)
                    if (!thinning || q + j >= L || sq[q] != sq[q + j]) m |= 1ull << q;
                sh.NE[tid][j - 1] = m;
            }
        }
        __syncthreads();

        const u32 T = sh.vbase[ng];
        const u64 base_out = COUNT_ONLY ? 0ull : P.rec_off[gid0];
        for (u32 rb = 0; rb < T; rb += GEN_THREADS * GEN_R) {
            const u32 f0 = min(T, rb + tid * GEN_R), f1 = min(T, f0 + GEN_R);
            // ---- sweep 1: survivors of this thread's range ----
            u32 mine = 0, gcur = 0xffffffffu, gacc = 0;
            gen_walk(sh, f0, f1, ng, d, [&](u32 g, u32, int k, const int* p) {
                bool ok = gen_canonical(sh, g, k, p);
                if (CHUNKED && ok) ok = gen_in_chunk(gen_hash(sh, g, k, p), sh.len[g] - (u32)k, P.chunk_lo, P.chunk_hi);
                if (COUNT_ONLY) {
                    if (g != gcur) {
                        if (gacc) atomicAdd(&sh.cnt[gcur], gacc);
                        gcur = g, gacc = 0;
                    }
                    gacc += ok ? 1u : 0u;
                }
                mine += ok ? 1u : 0u;
            });
            if (COUNT_ONLY) {
                if (gacc) atomicAdd(&sh.cnt[gcur], gacc);
                continue;
            }
            // ---- block exclusive scan of the survivor counts ----
            u32 inc = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u32 t = __shfl_up_sync(SD_FULL, inc, o);
                if (lane >= (u32)o) inc += t;
            }
            if (lane == 31) sh.wtot[warp] = inc;
            __syncthreads();
            u32 woff = sh.running, all = 0;
#pragma unroll
            for (int w = 0; w < GEN_NW; ++w) {
                const u32 c = sh.wtot[w];
                if ((u32)w < warp) woff += c;
                all += c;
            }
            __syncthreads();
            if (tid == 0) sh.running += all;
            // ---- sweep 2: hash and write ----
            u64* out = P.records + base_out + woff + inc - mine;
            gen_walk(sh, f0, f1, ng, d, [&](u32 g, u32, int k, const int* p) {
                if (!gen_canonical(sh, g, k, p)) return;
                const u64 h = gen_hash(sh, g, k, p);
                if (CHUNKED && !gen_in_chunk(h, sh.len[g] - (u32)k, P.chunk_lo, P.chunk_hi)) return;
                const u64 key = h >> kshift;
                *out++ = (key << P.id_bits) | (gid0 + g);
                for (int ps = 0; ps < P.npass; ++ps) atomicAdd(&s_hist[ps * 256 + ((u32)(key >> (P.hshift + 8 * ps)) & 255u)], 1u);
            });
        }
        __syncthreads();
        if (COUNT_ONLY) {
            if (tid < ng) P.cnt[gid0 + tid] = sh.cnt[tid];
        } else if (tid == 0) {
            if ((u64)sh.running != P.rec_off[gid0 + ng] - base_out) atomicOr(&P.info->err, (u32)SD_ERR_INTERNAL);
        }
    }
    if (!COUNT_ONLY) {
        __syncthreads();
        for (int i = tid; i < P.npass * 256; i += GEN_THREADS)
            if (s_hist[i]) atomicAdd(&P.ghist[i], s_hist[i]);
    }
}

// ---------------------------------------------------------------------------------------------
// Fast path (d <= 2, longest sequence <= 32): one warp per batch of consecutive sequences packed into
// its 32 lanes, lane = residue position.  The pairs {p1 < p2} of a length-L sequence are enumerated as
// {a, (a + delta) mod L} for delta = 1 .. (L-1)/2 (plus half a round at delta = L/2 when L is even):
// every lane of a sequence does the same number of rounds, no unranking, no search.  Per sequence the
// warp keeps U[p] = A[p] - Binv*A[p+1] and V[p] = Binv*U[p] in shared memory, so that
//     H({})      = A[L]                              + (L+1)*K
//     H({p})     = U[p]         + Binv*A[L]          + L*K
//     H({p1,p2}) = U[p1] + V[p2] + Binv^2*A[L]       + (L-1)*K
// (the same function as the general path) costs two shared loads and two adds per variant.
// The leftmost-embedding rule needs two ballots per batch: canon1 (s[p] != s[p+1] or p last) and
// adjok (the adjacent pair {p, p+1} is canonical); a non-adjacent pair is canonical iff both ends are.
// Without chunking the record count has the closed form
//     1 + B + B(B-1)/2 - #{p: canon1[p] & canon1[p+1]} + #adjok,   B = popcount(canon1)
// so the count pass never enters the delta loop.
constexpr int G2_THREADS = 256, G2_NW = G2_THREADS / 32;

struct Gen2Shared {
    u64 U[G2_NW][32];
    u64 V[G2_NW][32];
    u64 R[32];
    u64 Bpow[33];
    unsigned char map[G2_NW][32];
};

// One emission round of the fast path: lanes with `valid` append (hash, id) to their sequence's
// record range (rank by ballot inside the sequence's lane segment) and count the key's digits.
template <bool COUNT_ONLY, bool CHUNKED, int NPASS>
__device__ __forceinline__ void g2_emit(bool valid, u64 h, u32 vlen, const GenParams& P, u32 segmask, u32 lane_lt, u64 gid,
                                        int kshift, u64*& out, u32& run, u32* s_hist) {
    if (CHUNKED) valid = valid && gen_in_chunk(h, vlen, P.chunk_lo, P.chunk_hi);
    const u32 bal = __ballot_sync(SD_FULL, valid) & segmask;
    if (!COUNT_ONLY) {
        if (valid) {
            const u64 key = h >> kshift;
            out[__popc(bal & lane_lt)] = (key << P.id_bits) | gid;
            if (NPASS > 0) {
#pragma unroll
                for (int ps = 0; ps < NPASS; ++ps) atomicAdd(&s_hist[ps * 256 + ((u32)(key >> (P.hshift + 8 * ps)) & 255u)], 1u);
            } else {
                for (int ps = 0; ps < P.npass; ++ps) atomicAdd(&s_hist[ps * 256 + ((u32)(key >> (P.hshift + 8 * ps)) & 255u)], 1u);
            }
        }
        out += __popc(bal);
    }
    run += __popc(bal);
}

template <bool COUNT_ONLY, bool CHUNKED, int NPASS>
__global__ void __launch_bounds__(G2_THREADS) k_gen2(GenParams P) {
    extern __shared__ __align__(16) unsigned char gen_smem[];
    Gen2Shared& sh = *reinterpret_cast<Gen2Shared*>(gen_smem);
    u32* s_hist = reinterpret_cast<u32*>(gen_smem + sizeof(Gen2Shared));
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 lane_lt = (1u << lane) - 1u;
    if (tid < 32) sh.R[tid] = c_R[tid];
    if (tid < 33) sh.Bpow[tid] = c_Bpow[tid];
    if (!COUNT_ONLY)
        for (int i = tid; i < P.npass * 256; i += G2_THREADS) s_hist[i] = 0;
    __syncthreads();
    const int d = P.d;
    const bool thinning = P.thinning != 0;
    const u64 binv1 = c_Binv[1], binv2 = c_Binv[2];
    const int kshift = 64 - P.hash_bits;
    u64* const Uw = sh.U[warp];
    u64* const Vw = sh.V[warp];

    // warp task = 32 consecutive sequences of one set; groups_* count warp tasks here
    for (i64 wt = (i64)blockIdx.x * G2_NW + warp; wt < P.groups_total; wt += (i64)gridDim.x * G2_NW) {
        const bool in_b = wt >= P.groups_a;
        const SeqSetDev& S = in_b ? P.b : P.a;
        const i64 first = (in_b ? wt - P.groups_a : wt) * 32;
        const u32 ns = (u32)min((i64)32, S.n - first);
        const u64 gid0 = (u64)first + (in_b ? (u64)P.n_a : 0ull);
        i64 o0 = 0;
        u32 Li = 0;
        if (lane < ns) {
            o0 = S.off[first + lane];
            Li = min((u32)(S.off[first + lane + 1] - o0), P.prefix);
        }
        u32 cum_incl = Li;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 t = __shfl_up_sync(SD_FULL, cum_incl, o);
            if (lane >= (u32)o) cum_incl += t;
        }
        const u32 cum_excl = cum_incl - Li;
        u64 rec_base_i = 0;
        if (!COUNT_ONLY && lane < ns) rec_base_i = P.rec_off[gid0 + lane];

        u32 s = 0;
        while (s < ns) {
            const u32 base = __shfl_sync(SD_FULL, cum_excl, s);
            const u32 fit = __ballot_sync(SD_FULL, lane >= s && lane < ns && (cum_incl - base) <= 32u);
            const u32 e = s + __popc(fit);
            const u32 total = __shfl_sync(SD_FULL, cum_incl, e - 1) - base;
            const bool mine = lane >= s && lane < e;  // lane as SEQUENCE index of this batch
            // ---- empty sequences: one record (the empty variant) each ----
            if (mine && Li == 0) {
                const u64 h = K_LEN;  // A[L] = 0, (L + 1) * K
                const bool ok = !CHUNKED || gen_in_chunk(h, 0, P.chunk_lo, P.chunk_hi);
                if (COUNT_ONLY) {
                    P.cnt[gid0 + lane] = ok ? 1u : 0u;
                } else if (ok) {
                    const u64 key = h >> kshift;
                    P.records[rec_base_i] = (key << P.id_bits) | (gid0 + lane);
                    for (int ps = 0; ps < P.npass; ++ps) atomicAdd(&s_hist[ps * 256 + ((u32)(key >> (P.hshift + 8 * ps)) & 255u)], 1u);
                }
            }
            if (total > 0) {
                // ---- lane as POSITION: which sequence, which offset inside it ----
                const u32 hbit = (mine && Li > 0) ? (1u << (cum_excl - base)) : 0u;
                const u32 heads = __reduce_or_sync(SD_FULL, hbit);
                if (mine && Li > 0) sh.map[warp][cum_excl - base] = (unsigned char)lane;
                __syncwarp();
                const bool active = lane < total;
                const u32 seg_start = active ? (31u - __clz(heads & (0xffffffffu >> (31u - lane)))) : 0u;
                const u32 si = active ? sh.map[warp][seg_start] : 0u;  // sequence index within the task
                const u32 Lsrc = __shfl_sync(SD_FULL, Li, si);
                const u32 L = active ? Lsrc : 0u;  // idle lanes: L = 0 switches every later predicate off
                const u64 rec_base = __shfl_sync(SD_FULL, rec_base_i, si);
                const u32 a = lane - seg_start;
                const u64 gid = gid0 + si;
                const u32 segmask = active ? (((L == 32u) ? 0xffffffffu : ((1u << L) - 1u)) << seg_start) : 0u;
                const i64 osrc = __shfl_sync(SD_FULL, o0, si);  // (all lanes take part: never inside the ternary)
                const u32 c = active ? ((u32)(unsigned char)S.seqs[osrc + a] & 31u) : 0u;
                const u32 cn = __shfl_down_sync(SD_FULL, c, 1), cnn = __shfl_down_sync(SD_FULL, c, 2);
                const bool has1 = a + 1 < L, has2 = a + 2 < L;
                const bool canon1 = active && (!thinning || !has1 || c != cn);
                const bool adjok = active && has1 && (!thinning || !has2 || (c != cnn && cn != cnn));
                const u32 m1 = __ballot_sync(SD_FULL, canon1), madj = __ballot_sync(SD_FULL, adjok);

                u32 run = 0;  // records of this lane's sequence so far (uniform inside a segment)
                if (COUNT_ONLY && !CHUNKED) {
                    const u32 B = __popc(m1 & segmask);
                    run = 1;
                    if (d >= 1) run += B;
                    if (d >= 2) {
                        const u32 inner = segmask & (segmask >> 1);  // positions p with p + 1 inside the segment
                        run += B * (B - 1) / 2 - __popc(m1 & (m1 >> 1) & inner) + __popc(madj & segmask);
                    }
                } else {
                    // ---- prefix hashes of the source sequences (segmented scan over lanes) ----
                    const u64 term = active ? sh.R[c] * sh.Bpow[a] : 0ull;
                    u64 aincl = term;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const u64 t = __shfl_up_sync(SD_FULL, aincl, o);
                        if (a >= (u32)o) aincl += t;
                    }
                    const u64 aexcl = aincl - term;
                    const u64 AL = __shfl_sync(SD_FULL, aincl, active ? seg_start + L - 1 : 0);
                    const u64 Uv = aexcl - binv1 * aincl;
                    Uw[lane] = Uv;
                    Vw[lane] = binv1 * Uv;
                    __syncwarp();
                    const u64 C0 = AL + (u64)(L + 1) * K_LEN;
                    const u64 C1 = binv1 * AL + (u64)L * K_LEN;
                    const u64 C2 = binv2 * AL + (u64)(L - 1) * K_LEN;
                    u64* out = P.records + rec_base;

                    g2_emit<COUNT_ONLY, CHUNKED, NPASS>(active && a == 0, C0, L, P, segmask, lane_lt, gid, kshift, out, run, s_hist);
                    if (d >= 1)
                        g2_emit<COUNT_ONLY, CHUNKED, NPASS>(canon1, Uv + C1, L - 1, P, segmask, lane_lt, gid, kshift, out, run, s_hist);
                    if (d >= 2) {
                        const u32 half = __reduce_max_sync(SD_FULL, L >> 1);
                        const u32 m1s = m1 >> seg_start, madjs = madj >> seg_start;  // segment-relative masks
                        const u64* const Us = Uw + seg_start;
                        const u64* const Vs = Vw + seg_start;
                        for (u32 dl = 1; dl <= half; ++dl) {
                            u32 b = a + dl;
                            b = (b >= L) ? b - L : b;
                            const u32 p1 = min(a, b) & 31u, p2 = max(a, b) & 31u;
                            const bool on = (2 * dl < L) || (2 * dl == L && a < dl);  // false on idle lanes (L = 0)
                            const u32 both = (m1s >> p1) & (m1s >> p2);
                            const u32 t = (p2 - p1 == 1u) ? (madjs >> p1) : both;
                            const u64 h = Us[p1] + Vs[p2] + C2;
                            g2_emit<COUNT_ONLY, CHUNKED, NPASS>(on && (t & 1u), h, L - 2, P, segmask, lane_lt, gid, kshift, out, run,
                                                                s_hist);
                        }
                    }
                    __syncwarp();  // U/V/map are reused by the next batch
                }
                if (active && a == 0) {
                    if (COUNT_ONLY) P.cnt[gid] = run;
                    else if ((u64)run != P.rec_off[gid + 1] - rec_base) atomicOr(&P.info->err, (u32)SD_ERR_INTERNAL);
                }
            }
            s = e;
        }
    }
    if (!COUNT_ONLY) {
        __syncthreads();
        for (int i = tid; i < P.npass * 256; i += G2_THREADS)
            if (s_hist[i]) atomicAdd(&P.ghist[i], s_hist[i]);
    }
}

// ---------------------------------------------------------------------------------------------
// Fused fast path: generation + level-1 partition (k_gen2_part).  Same enumeration and hash as k_gen2,
// but a record is not written in id order: it is staged in shared memory under the top 8 bits of its
// hash (GP_S slots per digit; one shared-memory atomic returns its slot) and the block flushes the
// stage to 256 global BINS of fixed capacity `cap1` (one global atomic per digit and flush claims the
// segment; each digit's records leave as one contiguous store).  No count pass, no offsets, no
// histogram: the order of the records inside a bin is irrelevant to the join.  A record that finds its
// digit's slots full goes straight to its bin (one global atomic).  A bin that would overflow raises
// info->part_overflow: the host then redoes the chunk with the exact (histogram-based) pipeline.
// (values swept on config 3 / config 5 in round 1: 512 threads, 2 or 4 resident blocks, rounds of 3600 / 7200 records
//  and flush thresholds from 2000 to 4500 all landed within 3 % of these)
constexpr int GP_THREADS = 256;    // threads per block (512 with two resident blocks: +2 %)
constexpr int GP_MINB = 3;         // resident blocks per SM (64 KB stage each)
constexpr int GP_FLUSH_AT = 2800;  // flush when more than this is staged after a round (i.e. after nearly every full round)
constexpr int GP_OVF = 64;         // overflow list entries
constexpr int GP_TRIP = 8;         // d = 3: (g1, g2) iterations per step of a batch (more, smaller units per round even the warps out: config 5 with 4 / 8 / 16 / 32: 1.40 / 1.33 / 1.41 / 1.58 ms)
constexpr int GP_ROUND = 5400;     // records a block stages per round (21 per digit of the 32 slots); the host turns it into batches per warp
                                   // (round 2: rounds of 3,300 records cost +10 %, i.e. ~2.3 us per flush stay exposed; 22 slots with four resident blocks: +7 %)
constexpr int GP_NW = GP_THREADS / 32, GP_S = 32;  // (16 slots per digit and 4-5 resident blocks: generation 0.66 -> 0.85-1.25 ms on config 3, the digits overflow)
static_assert(GP_THREADS == 256 && GP_S <= 32, "one thread per digit in the flush, one lane per slot of a row");

constexpr int GP_ROW = GP_S + 1;  // stage row stride in records: rank r of digit dg sits in 8-byte word dg * 33 + r, i.e. bank pair (dg + r) mod 16 — ranks are alike across digits, the odd stride spreads them
struct GenPartShared {
    u64 stage[256 * GP_ROW];
    // per warp, for the sequence whose first lane is s0 and whose length is L: W[2 * s0 + j] = V[j] for j < L and U[j - L]
    // for L <= j < 2L — the partner (a + dl) mod L of position a is ONE load at index a + dl, no wrap arithmetic
    u64 W[GP_NW][64];
    u64 R[32];
    u64 Bpow[33];
    u32 cnt[256];     // BYTES staged per digit since the last flush (8 per record; may exceed 8 * GP_S: the excess went to the overflow list)
    u32 gofs[256];    // flush: index of the claimed segment in bins (0xffffffff = bin full)
    u32 total[3];     // D3: records staged in round r go to total[r % 3] (three words: a fast warp of round r + 1 never touches the word the slow warps of round r still read)
    u32 novf;         // records in ovf[] (may count past GP_OVF: those went to the bins directly)
    u64 ovf[GP_OVF];  // records whose digit had no free slot: placed at the next flush (near-identical neighbouring sequences — clonal lineages — push the same digits in bursts)
    unsigned char map[GP_NW][32];
};
static_assert(sizeof(GenPartShared) <= (233472 - GP_MINB * 1024) / GP_MINB, "GP_MINB blocks per SM");

struct GenPartParams {
    GenParams g;
    u64* bins;    // 256 bins of cap1 records (256 * cap1 < 2^32)
    u32* cur;     // 256 bin cursors (zeroed by the host)
    u32 cap1;
    u32 batches;  // k_gen2_part: batches per warp and round
    i64 task_begin, task_end;  // k_gen2_part: the warp tasks of this launch — a slice when the input arrives in slices
    u32 task_seqs;             // k_gen2_part: consecutive sequences per warp task (a power of two <= 32; g.groups_* count tasks of this size)
};

// D3 (d == 3): the triples {p1 < p2 < p3} follow the pairs.  A triple is the three points a, a + g1, a + g1 + g2
// on the circle of L positions with gaps (g1, g2, g3 = L - g1 - g2); of its three starting points exactly one is
// kept: the one whose LAST gap is the largest (g3 > g1 and g3 >= g2; all gaps equal: a < g1) — so every lane of a
// sequence enumerates the same (g1, g2) and the work is balanced.  H = U[p1] + V[p2] + Binv * V[p3] + C3.  The
// leftmost-embedding rule is the bit-mask test of gen_canonical on segment-relative masks.  A batch then makes
// thousands of records, so it is RESUMABLE: step 0 = everything up to the pairs, step g1 = the triples of that
// first gap; the block's flush decision falls between steps.
template <bool CHUNKED, bool PLAIN, bool D3>
__global__ void __launch_bounds__(GP_THREADS, GP_MINB) k_gen2_part(GenPartParams PP) {
    extern __shared__ __align__(16) unsigned char gen_smem[];
    GenPartShared& sh = *reinterpret_cast<GenPartShared*>(gen_smem);
    const GenParams& P = PP.g;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 32) sh.R[tid] = c_R[tid];
    if (tid < 33) sh.Bpow[tid] = c_Bpow[tid];
    if (tid < 256) sh.cnt[tid] = 0;
    if (tid < 3) sh.total[tid] = 0;
    if (tid == 0) sh.novf = 0;
    __syncthreads();
    const int d = P.d;
    const bool thinning = P.thinning != 0;
    const u64 binv1 = c_Binv[1], binv2 = c_Binv[2];
    const int kshift = 64 - P.hash_bits, id_bits = P.id_bits;  // PLAIN: kshift == id_bits, the record is the hash with its low id_bits replaced by the id
    const u32 idmask_lo = id_bits >= 32 ? 0xffffffffu : ((1u << id_bits) - 1u);
    // shared-window addresses of the counters and the stage, computed once and kept in registers (left to itself the
    // compiler re-derives them from SR_CgaCtaId at every use: three instructions per record)
    u32 cnt_sa = (u32)__cvta_generic_to_shared(sh.cnt), stage_sa = (u32)__cvta_generic_to_shared(sh.stage);
    asm volatile("" : "+r"(cnt_sa), "+r"(stage_sa));
    u64* const Ww = sh.W[warp];
    u32 made = 0;  // D3: records this lane staged since the warp last reported

    // one record: its digit's counter (in bytes) hands out the slot; rank r of digit dg -> byte dg * 264 + 8 r of the stage
    const u64 ch_lo = P.chunk_lo, ch_hi = P.chunk_hi;
    auto push1 = [&](u64 h, u64 gid, u32 vlen) {
        if (CHUNKED && !gen_in_chunk(h, vlen, ch_lo, ch_hi)) return;
        const u32 dg = (u32)(h >> 56);
        u64 rec;
        if (PLAIN) rec = ((u64)(u32)(h >> 32) << 32) | (((u32)h & ~idmask_lo) | (u32)gid);  // id_bits <= 31 here
        else rec = ((h >> kshift) << id_bits) | gid;
        u32 r8;  // plain ATOMS.ADD with return (no compiler-inserted aggregation)
        asm volatile("atom.shared.add.u32 %0, [%1], 8;" : "=r"(r8) : "r"(cnt_sa + dg * 4u) : "memory");
        const u32 row = stage_sa + dg * (u32)(GP_ROW * 8);
        if (r8 < (u32)(GP_S * 8)) {
            asm volatile("st.shared.u64 [%0], %1;" ::"r"(row + r8), "l"(rec) : "memory");
        } else {
            const u32 o = atomicAdd(&sh.novf, 1u);
            if (o < (u32)GP_OVF) {
                sh.ovf[o] = rec;
            } else {
                const u32 at = atomicAdd(&PP.cur[dg], 1u);
                if (at < PP.cap1) PP.bins[(u64)dg * PP.cap1 + at] = rec;
                else atomicOr(&P.info->part_overflow, 1u);
            }
        }
        if (D3) ++made;
    };
    auto push = [&](bool valid, u64 h, u64 gid, u32 vlen) {
        if (valid) push1(h, gid, vlen);
    };

    // warp task = 32 consecutive sequences of one set, cut into batches that fill the 32 lanes; the block
    // advances `batches` batches per warp and round, then flushes
    // (the warps of a block take tasks far apart in the input: neighbouring sequences are often near-identical —
    // clonal lineages — and would all push the same digits at the same time)
    i64 wt = PP.task_begin + (i64)warp * gridDim.x + blockIdx.x;
    const i64 wstride = (i64)gridDim.x * GP_NW;
    bool have = false;  // a task is loaded and has batches left
    bool is_empty = false;  // lane as sequence index: a sequence of length 0 (its one record is the empty variant)
    u32 rnd = 0, staged = 0;  // D3: round index mod 3; records staged since the last flush (block-uniform)
    u32 s = 0, ns = 0, Li = 0, cum_incl = 0, cum_excl = 0;
    u64 gid0 = 0;
    i64 o0 = 0;  // lane as sequence index: offset of its residues
    const int8_t* seqs = nullptr;
    // D3: the state of a batch between its steps
    u32 step = 0, t_g2 = 1, t_a = 0, t_L = 0, t_seg = 0, t_e = 0, t_g1max = 0, t_ne1 = 0, t_ne2 = 0, t_ne3 = 0, t_Lmax = 0;
    u64 t_gid = 0, t_C3 = 0;
    while (true) {
#pragma unroll 1
        for (u32 rep = 0; rep < PP.batches; ++rep) {  // the same trip count in every warp: rounds stay balanced
        if (!have && wt < PP.task_end) {
            const bool in_b = wt >= P.groups_a;
            const SeqSetDev& S = in_b ? P.b : P.a;
            const i64 first = (in_b ? wt - P.groups_a : wt) * (i64)PP.task_seqs;
            ns = (u32)min((i64)PP.task_seqs, S.n - first);
            gid0 = (u64)first + (in_b ? (u64)P.n_a : 0ull);
            seqs = S.seqs;
            o0 = 0;
            Li = 0;
            if (lane < ns) {
                o0 = S.off[first + lane];
                Li = min((u32)(S.off[first + lane + 1] - o0), P.prefix);
            }
            is_empty = lane < ns && Li == 0;
            if (CHUNKED) {
                // a sequence none of whose deletion depths reaches into this chunk takes no lanes at all
                bool rel = false;
                for (int k = 0; k <= d; ++k) rel = rel || (Li >= (u32)k && gen_len_in_chunk(Li - (u32)k, ch_lo, ch_hi));
                if (!rel) Li = 0, is_empty = false;
            }
            cum_incl = Li;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u32 t = __shfl_up_sync(SD_FULL, cum_incl, o);
                if (lane >= (u32)o) cum_incl += t;
            }
            cum_excl = cum_incl - Li;
            s = 0;
            have = true;
            wt += wstride;
        }
        if (D3 && have && step > 0) {
            // ---- one step of a batch's triples: GP_TRIP (g1, g2) iterations from where the last step stopped, so
            //      that a step costs every warp the same whatever its sequence lengths ----
            const u32 a = t_a, L = t_L;
            const u32 v_sa = (u32)__cvta_generic_to_shared(Ww + 2 * t_seg), u_sa = v_sa + 8u * L;
            for (u32 it = 0; it < (u32)GP_TRIP && step <= t_g1max; ++it) {
                const u32 g1 = step, g2 = t_g2;
                const u32 g2hi = min((t_Lmax - g1) >> 1, t_Lmax - 2 * g1);  // g3 >= g2 and g3 > g1 (or all equal) at the longest length
                const u32 g3 = L - g1 - g2;  // meaningless (huge) where g1 + g2 >= L: `ok` is false there
                const bool ok = g1 + g2 < L && ((g3 > g1 && g3 >= g2) || (g1 == g2 && g2 == g3 && a < g1));
                u32 y = a + g1, z = y + g2;
                const bool wy = y >= L, wz = z >= L;
                y = (wy ? y - L : y) & 31u;
                z = (wz ? z - L : z) & 31u;
                // sorted positions: no wrap (a, y, z); z wrapped (z, a, y); both wrapped (y, z, a)
                const u32 p1 = wy ? y : (wz ? z : a), p2 = wy ? z : (wz ? a : y), p3 = wy ? a : (wz ? y : z);
                const u32 D = (1u << a) | (1u << y) | (1u << z);
                const u32 r2 = D & (D >> 1), r3 = r2 & (D >> 2);
                const u32 bad = ((D & ~r2) & ~t_ne1) | ((r2 & ~r3) & ~t_ne2) | (r3 & ~t_ne3);
                u64 u1, v2, v3;
                asm volatile("ld.shared.u64 %0, [%1];" : "=l"(u1) : "r"(u_sa + p1 * 8u));
                asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v2) : "r"(v_sa + p2 * 8u));
                asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v3) : "r"(v_sa + p3 * 8u));
                push(g2 <= g2hi && ok && bad == 0, u1 + v2 + binv1 * v3 + t_C3, t_gid, L - 3u);
                if (g2 >= g2hi) {
                    ++step;
                    t_g2 = 1;
                } else {
                    ++t_g2;
                }
            }
            if (step > t_g1max) {
                step = 0;
                __syncwarp();  // W/map are reused by the next batch
                s = t_e;
                have = s < ns;
            }
            const u32 wmade = __reduce_add_sync(SD_FULL, made);
            made = 0;
            if (lane == 0 && wmade) atomicAdd(&sh.total[rnd], wmade);
        } else if (have) {
            // ---- one batch: sequences [s, e) of the task ----
            const u32 base = __shfl_sync(SD_FULL, cum_excl, s);
            const u32 fit = __ballot_sync(SD_FULL, lane >= s && lane < ns && (cum_incl - base) <= 32u);
            const u32 e = s + __popc(fit);
            const u32 total = __shfl_sync(SD_FULL, cum_incl, e - 1) - base;
            const bool mine = lane >= s && lane < e;  // lane as SEQUENCE index of this batch
            if (mine && is_empty) push(true, K_LEN, gid0 + lane, 0u);  // the empty variant of an empty sequence
            if (total > 0) {
                // ---- lane as POSITION: which sequence, which offset inside it ----
                const u32 hbit = (mine && Li > 0) ? (1u << (cum_excl - base)) : 0u;
                const u32 heads = __reduce_or_sync(SD_FULL, hbit);
                if (mine && Li > 0) sh.map[warp][cum_excl - base] = (unsigned char)lane;
                __syncwarp();
                const bool active = lane < total;
                const u32 seg_start = active ? (31u - __clz(heads & (0xffffffffu >> (31u - lane)))) : 0u;
                const u32 si = active ? sh.map[warp][seg_start] : 0u;
                const u32 Lsrc = __shfl_sync(SD_FULL, Li, si);
                const u32 L = active ? Lsrc : 0u;  // idle lanes: L = 0 switches every later predicate off
                const u32 a = lane - seg_start;
                const u64 gid = gid0 + si;
                const i64 osrc = __shfl_sync(SD_FULL, o0, si);  // (all lanes take part: never inside the ternary)
                const u32 c = active ? ((u32)(unsigned char)seqs[osrc + a] & 31u) : 0u;
                const u32 cn = __shfl_down_sync(SD_FULL, c, 1), cnn = __shfl_down_sync(SD_FULL, c, 2);
                const bool has1 = a + 1 < L, has2 = a + 2 < L;
                const bool canon1 = active && (!thinning || !has1 || c != cn);
                const bool adjok = active && has1 && (!thinning || !has2 || (c != cnn && cn != cnn));
                const u32 m1 = __ballot_sync(SD_FULL, canon1), madj = __ballot_sync(SD_FULL, adjok);
                // ---- prefix hashes of the source sequences (segmented scan over lanes) ----
                const u64 term = active ? sh.R[c] * sh.Bpow[a] : 0ull;
                u64 aincl = term;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u64 t = __shfl_up_sync(SD_FULL, aincl, o);
                    if (a >= (u32)o) aincl += t;
                }
                const u64 aexcl = aincl - term;
                const u64 AL = __shfl_sync(SD_FULL, aincl, active ? seg_start + L - 1 : 0);
                const u64 Uv = aexcl - binv1 * aincl;
                if (active) {  // (2 * seg_start + 2L <= 64: the batch holds at most 32 residues)
                    Ww[2 * seg_start + a] = binv1 * Uv;
                    Ww[2 * seg_start + L + a] = Uv;
                }
                __syncwarp();
                // chunked: only the deletion depths whose variant length reaches into this chunk are enumerated
                const bool in0 = !CHUNKED || gen_len_in_chunk(L, ch_lo, ch_hi), in1 = !CHUNKED || gen_len_in_chunk(L - 1u, ch_lo, ch_hi);
                const bool in2 = !CHUNKED || (L >= 2u && gen_len_in_chunk(L - 2u, ch_lo, ch_hi));
                push(active && a == 0 && in0, AL + (u64)(L + 1) * K_LEN, gid, L);
                if (d >= 1) push(canon1 && in1, Uv + binv1 * AL + (u64)L * K_LEN, gid, L - 1u);
                if (d >= 2) {
                    // pairs {a, (a + dl) mod L}: lane a runs dl = 1 .. dlmax (every unordered pair once); the
                    // partner b sits after a (no wrap: H = U[a] + V[b]) or before it (wrap: H = U[b] + V[a])
                    const u64 C2 = binv2 * AL + (u64)(L - 1) * K_LEN;
                    const u64 UC = Uv + C2, VC = binv1 * Uv + C2;
                    const u32 half = __reduce_max_sync(SD_FULL, in2 ? L >> 1 : 0u);
                    const u32 dlmax = active ? ((L - 1) >> 1) + (((L & 1u) == 0u && a < (L >> 1)) ? 1u : 0u) : 0u;
                    const u32 m1s = m1 >> seg_start;  // segment-relative mask
                    // vmask bit dl: the pair {a, (a + dl) mod L} makes a record.  dl >= 2: both members are canonical
                    // single deletions; dl = 1: the adjacent pair {a, a + 1} has its own rule, the wrapped pair
                    // {0, L - 1} is adjacent only if L == 2
                    const u32 m1L = L >= 32u ? m1s : (m1s & ((1u << L) - 1u));
                    const u32 rot = (u32)((((u64)m1L << L) | (u64)m1L) >> a);  // bit dl = m1s bit (a + dl) mod L
                    const bool wrap1 = a + 1 >= L;
                    const bool ok1 = wrap1 ? (L == 2u ? ((madj >> seg_start) & 1u) != 0u : (canon1 && (m1s & 1u))) : adjok;
                    u32 vmask = (canon1 ? rot : 0u) & ((2u << dlmax) - 1u) & ~3u;
                    if (ok1 && dlmax >= 1u) vmask |= 2u;
                    if (!in2) vmask = 0u;
                    const u32 wth = L - a;  // dl >= wth: the partner wrapped
                    const u32 w_sa = (u32)__cvta_generic_to_shared(Ww + 2 * seg_start + a);
                    u64 UCr = UC, VCr = VC;
                    asm volatile("" : "+l"(UCr), "+l"(VCr));  // both in registers (else the wrap select is re-derived as a 64-bit multiply per record)
                    u32 vm = __brev(vmask) << 1;  // bit 31 = dl 1: the sign tells whether this lane has a record
#pragma unroll 4
                    for (u32 dl = 1; dl <= half; ++dl, vm <<= 1) {
                        if ((int)vm < 0) {
                            u64 o;
                            asm volatile("ld.shared.u64 %0, [%1];" : "=l"(o) : "r"(w_sa + dl * 8u));
                            push1(o + (dl >= wth ? VCr : UCr), gid, L - 2u);
                        }
                    }
                }
                if (D3) {  // the triples follow, one first gap per step
                    const u32 cnnn = __shfl_down_sync(SD_FULL, c, 3);
                    const bool ne2 = active && (!thinning || !has2 || c != cnn);
                    const bool ne3 = active && (!thinning || !(a + 3 < L) || c != cnnn);
                    const u32 b2 = __ballot_sync(SD_FULL, ne2), b3 = __ballot_sync(SD_FULL, ne3);
                    const bool in3 = !CHUNKED || (L >= 3u && gen_len_in_chunk(L - 3u, ch_lo, ch_hi));
                    t_Lmax = __reduce_max_sync(SD_FULL, in3 ? L : 0u);
                    t_g1max = t_Lmax >= 3 ? (t_Lmax - 1) >> 1 : 0;
                    t_a = a, t_L = in3 ? L : 0u, t_seg = seg_start, t_e = e, t_gid = gid;
                    t_ne1 = m1 >> seg_start, t_ne2 = b2 >> seg_start, t_ne3 = b3 >> seg_start;
                    t_C3 = binv1 * binv2 * AL + (u64)(L - 2) * K_LEN;
                    if (t_g1max > 0) step = 1, t_g2 = 1;
                }
                if (!D3 || step == 0) __syncwarp();  // W/map are reused by the next batch
            }
            if (!D3 || step == 0) {
                s = e;
                have = s < ns;
            }
            if (D3) {
                const u32 wmade = __reduce_add_sync(SD_FULL, made);
                made = 0;
                if (lane == 0 && wmade) atomicAdd(&sh.total[rnd], wmade);
            }
        }
        }
        // ---- round end: anyone left?  d <= 2: the host sized the round to fill the stage, flush.  D3: flush when the
        //      stage is about full (always at the end) ----
        const bool more = have || wt < PP.task_end;
        const int any_more = __syncthreads_or(more);
        bool flush = true;
        if (D3) {
            staged += sh.total[rnd];
            rnd = rnd == 2 ? 0 : rnd + 1;
            if (tid == 0) sh.total[rnd == 2 ? 0 : rnd + 1] = 0;  // the word of the round after next: nobody reads or adds to it now
            flush = staged > (u32)GP_FLUSH_AT || (!any_more && staged > 0);
        }
        if (flush) {
            const u32 novf = min(sh.novf, (u32)GP_OVF);  // (final since the round barrier; everyone has it before the next barrier, after which thread 0 clears the word)
            if (tid < 256) {
                const u32 cn_ = min(sh.cnt[tid] >> 3, (u32)GP_S);
                u32 g = 0;
                if (cn_) {
                    g = atomicAdd(&PP.cur[tid], cn_);
                    if (g + cn_ > PP.cap1) {
                        atomicOr(&P.info->part_overflow, 1u);
                        g = 0xffffffffu;
                    } else {
                        g += tid * PP.cap1;
                    }
                }
                sh.gofs[tid] = g;
            }
            __syncthreads();
            if (tid == 0) sh.novf = 0;
            static_assert(256 / GP_NW == 32, "a warp copies, then clears, 32 rows: one counter per lane");
            u64* const bins = PP.bins;
#pragma unroll 4
            for (u32 k = 0; k < 32; ++k) {
                const u32 dg = warp * 32 + k;
                const u32 g = sh.gofs[dg], cn_ = min(sh.cnt[dg] >> 3, (u32)GP_S);
                if (lane < cn_ && g != 0xffffffffu) bins[g + lane] = sh.stage[dg * GP_ROW + lane];
            }
            __syncwarp();
            sh.cnt[warp * 32 + lane] = 0;  // (after the claims only this warp reads these counters)
            for (u32 i = tid; i < novf; i += GP_THREADS) {  // the overflow records, one global atomic each
                const u64 rec = sh.ovf[i];
                const u32 dg = (u32)(rec >> (P.id_bits + P.hash_bits - 8)) & 255u;
                const u32 at = atomicAdd(&PP.cur[dg], 1u);
                if (at < PP.cap1) PP.bins[(u64)dg * PP.cap1 + at] = rec;
                else atomicOr(&P.info->part_overflow, 1u);
            }
            staged = 0;
            __syncthreads();  // rows, counters and the overflow list are free again
        }
        if (!any_more) break;
    }
}

// ---------------------------------------------------------------------------------------------
// Fused general path (k_generate_part): the enumeration of k_generate (any d <= 4, any length <= 64)
// with the staging / flushing of k_gen2_part.  One sweep per round instead of two: no counts, no scan,
// no offsets — a canonical deletion set is hashed and pushed under its top 8 hash bits.
constexpr int GQ_S = 16;          // stage slots per digit (16 or 32; 32 halves the resident blocks: slower on config 5 shapes)
constexpr int GQ_R = 8;           // consecutive deletion sets per thread and round: a round makes at most GEN_THREADS * GQ_R records
constexpr int GQ_MINB = 3;        // resident blocks per SM (one more with 32-residue table rows)
constexpr int GQ_FLUSH_AT = 900;  // flush when more than this is staged after a round
static_assert(GQ_S == 16 || GQ_S == 32, "flush copies 32 / GQ_S digits per warp instruction");

struct GenPartStage {
    u64 stage[256 * GQ_S];  // digit dg, rank r -> stage[dg * GQ_S + ((r + dg) & (GQ_S - 1))]
    u32 cnt[256];
    uint2 fl[256];
    u32 total[3];  // as in GenPartShared
};

template <bool CHUNKED, int LW>
__global__ void __launch_bounds__(GEN_THREADS, LW <= 32 ? GQ_MINB + 1 : GQ_MINB) k_generate_part(GenPartParams PP) {
    typedef GenSharedT<LW> SH;
    extern __shared__ __align__(16) unsigned char gen_smem[];
    SH& sh = *reinterpret_cast<SH*>(gen_smem);
    GenPartStage& ps = *reinterpret_cast<GenPartStage*>(gen_smem + ((sizeof(SH) + 15) & ~(size_t)15));
    const GenParams& P = PP.g;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < (SD_L_MAX + 1) * (SD_D_MAX + 1); i += GEN_THREADS) sh.binom[i] = c_binom[i];
    for (int i = tid; i < (SD_L_MAX + 1) * (SD_D_MAX + 2); i += GEN_THREADS) sh.vcum[i] = c_vcum[i];
    if (tid < 32) sh.R[tid] = c_R[tid];
    if (tid <= SD_L_MAX) sh.Bpow[tid] = c_Bpow[tid];
    ps.cnt[tid] = 0;
    if (tid < 3) ps.total[tid] = 0;
    u32 rnd = 0, staged = 0;
    const int d = P.d;
    const bool thinning = P.thinning != 0;
    const int kshift = 64 - P.hash_bits, id_bits = P.id_bits;
    const u32 cnt_sa = (u32)__cvta_generic_to_shared(ps.cnt);

    auto flush = [&]() {  // all threads; the caller has synchronised
        {
            const u32 cn_ = min(ps.cnt[tid], (u32)GQ_S);
            u32 g = 0;
            if (cn_) {
                g = atomicAdd(&PP.cur[tid], cn_);
                if (g + cn_ > PP.cap1) {
                    atomicOr(&P.info->part_overflow, 1u);
                    g = 0xffffffffu;
                } else {
                    g += tid * PP.cap1;
                }
            }
            ps.fl[tid] = make_uint2(g, g == 0xffffffffu ? 0u : cn_);
        }
        __syncthreads();
        // 32 / GQ_S digits per warp instruction (GQ_S = 16: lanes 0-15 and 16-31)
        constexpr u32 DPW = 32 / GQ_S;
        for (u32 dg = DPW * warp + lane / GQ_S; dg < 256; dg += DPW * GEN_NW) {
            const uint2 f = ps.fl[dg];
            const u32 o = lane & (GQ_S - 1);
            if (o < f.y) PP.bins[f.x + o] = ps.stage[dg * GQ_S + ((o + dg) & (GQ_S - 1))];
        }
        __syncthreads();
        ps.cnt[tid] = 0;
        staged = 0;
        __syncthreads();
    };

    for (i64 gi = blockIdx.x; gi < P.groups_total; gi += gridDim.x) {
        const bool in_b = gi >= P.groups_a;
        const SeqSetDev& S = in_b ? P.b : P.a;
        const i64 first = (in_b ? gi - P.groups_a : gi) * GEN_G;
        const u32 ng = (u32)min((i64)GEN_G, S.n - first);
        const u64 gid0 = (u64)first + (in_b ? (u64)P.n_a : 0ull);
        __syncthreads();  // previous group fully consumed (also orders the table fill above)
        if (tid < GEN_G) {
            u32 L = 0;
            if (tid < ng) {
                const i64 a = S.off[first + tid];
                L = min((u32)(S.off[first + tid + 1] - a), P.prefix);
                sh.off[tid] = a;
            }
            sh.len[tid] = L;
            u32 v = tid < ng ? sh.vcum[L * (SD_D_MAX + 2) + d + 1] : 0, inc = v;  // V(L, d), scanned over the group
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u32 t = __shfl_up_sync(SD_FULL, inc, o);
                if (lane >= (u32)o) inc += t;
            }
            sh.vbase[tid + 1] = inc;
            if (tid == 0) sh.vbase[0] = 0;
        }
        __syncthreads();
        for (u32 idx = tid; idx < ng * (u32)P.width; idx += GEN_THREADS) {
            const u32 g = idx / (u32)P.width, q = idx - g * (u32)P.width;
            sh.seq[g][q] = q < sh.len[g] ? (unsigned char)S.seqs[sh.off[g] + q] : (unsigned char)0;
        }
        __syncthreads();
        if (tid < ng) {  // per-sequence tables (as in k_generate)
            const u32 L = sh.len[tid];
            const unsigned char* sq = sh.seq[tid];
            u64 acc = 0;
            for (u32 q = 0; q < L; ++q) {
                const u64 nxt = acc + sh.R[sq[q] & 31] * sh.Bpow[q];
                sh.U[tid][q] = acc - c_Binv[1] * nxt;
                acc = nxt;
            }
            for (int k = 0; k <= SD_D_MAX; ++k) sh.C[tid][k] = c_Binv[k] * acc + (u64)(L - k + 1) * K_LEN;
            for (int j = 1; j <= SD_D_MAX; ++j) {
                u64 m = 0;
                for (u32 q = 0; q < L; ++q)
                    if (!thinning || q + j >= L || sq[q] != sq[q + j]) m |= 1ull << q;
                sh.NE[tid][j - 1] = m;
            }
        }
        __syncthreads();

        const u32 T = sh.vbase[ng];
        for (u32 rb = 0; rb < T; rb += GEN_THREADS * GQ_R) {
            const u32 f0 = min(T, rb + tid * GQ_R), f1 = min(T, f0 + GQ_R);
            u32 made = 0;
            gen_walk(sh, f0, f1, ng, d, [&](u32 g, u32, int k, const int* p) {
                if (!gen_canonical(sh, g, k, p)) return;
                const u64 h = gen_hash(sh, g, k, p);
                if (CHUNKED && !gen_in_chunk(h, sh.len[g] - (u32)k, P.chunk_lo, P.chunk_hi)) return;
                const u32 dg = (u32)(h >> 56);
                const u64 rec = ((h >> kshift) << id_bits) | (gid0 + g);
                u32 r;
                asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(r) : "r"(cnt_sa + dg * 4u) : "memory");
                if (r < (u32)GQ_S) {
                    ps.stage[dg * GQ_S + ((r + dg) & (GQ_S - 1))] = rec;
                } else {
                    const u32 at = atomicAdd(&PP.cur[dg], 1u);
                    if (at < PP.cap1) PP.bins[(u64)dg * PP.cap1 + at] = rec;
                    else atomicOr(&P.info->part_overflow, 1u);
                }
                ++made;
            });
            const u32 wmade = __reduce_add_sync(SD_FULL, made);
            if (lane == 0 && wmade) atomicAdd(&ps.total[rnd], wmade);
            __syncthreads();
            staged += ps.total[rnd];
            rnd = rnd == 2 ? 0 : rnd + 1;
            if (tid == 0) ps.total[rnd == 2 ? 0 : rnd + 1] = 0;  // the word of the round after next
            if (staged > (u32)GQ_FLUSH_AT) flush();  // block-uniform
        }
    }
    __syncthreads();
    if (staged > 0) flush();
}

typedef void (*Gen2Kernel)(GenParams);
template <bool COUNT_ONLY>
Gen2Kernel gen2_pick(bool chunked, int npass) {
    if (chunked) return k_gen2<COUNT_ONLY, true, 0>;
    if (COUNT_ONLY) return k_gen2<COUNT_ONLY, false, 0>;
    switch (npass) {
        case 1: return k_gen2<COUNT_ONLY, false, 1>;
        case 2: return k_gen2<COUNT_ONLY, false, 2>;
        case 3: return k_gen2<COUNT_ONLY, false, 3>;
        default: return k_gen2<COUNT_ONLY, false, 0>;
    }
}

u64 splitmix64(u64& x) {
    u64 z = (x += 0x9e3779b97f4a7c15ull);
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
    return z ^ (z >> 31);
}

GenParams make_params(SeqSetDev a, SeqSetDev b, const Layout& lay, int width) {
    GenParams P{};
    P.a = a;
    P.b = b;
    P.n_a = a.n;
    P.groups_a = (a.n + GEN_G - 1) / GEN_G;
    P.groups_total = P.groups_a + (b.n + GEN_G - 1) / GEN_G;
    P.d = lay.d;
    P.width = width;
    P.thinning = lay.thinning;
    P.hash_bits = lay.hash_bits;
    P.id_bits = lay.id_bits;
    P.n_chunks = lay.n_chunks;
    P.chunk = lay.chunk;
    P.chunk_lo = lay.chunk_lo;
    P.chunk_hi = lay.chunk_hi;
    P.prefix = lay.prefix > 0 ? (u32)lay.prefix : (u32)SD_L_MAX;
    return P;
}

int gen_grid(i64 groups) { return (int)std::min<i64>(groups, 148 * 6); }

bool use_fast(const Layout& lay, int width) { return lay.d <= 2 && width - 1 <= 32 && !lay.force_general; }
// the fused lane-per-position generator also does d = 3
bool use_fast_part(const Layout& lay, int width) { return lay.d <= 3 && width - 1 <= 32 && !lay.force_general; }

GenParams make_params2(SeqSetDev a, SeqSetDev b, const Layout& lay, int width) {
    GenParams P = make_params(a, b, lay, width);
    P.groups_a = (a.n + 31) / 32;  // warp tasks of 32 sequences
    P.groups_total = P.groups_a + (b.n + 31) / 32;
    return P;
}
int gen2_grid(i64 wtasks) { return (int)std::min<i64>((wtasks + G2_NW - 1) / G2_NW, 148 * 8); }

// the fused generators: [d == 3][chunked][plain] and [narrow rows][chunked]
typedef void (*GenPartKernel)(GenPartParams);
const GenPartKernel GEN2_PART_KERNELS[8] = {k_gen2_part<false, false, false>, k_gen2_part<false, true, false>, k_gen2_part<true, false, false>,
                                            k_gen2_part<true, true, false>,  k_gen2_part<false, false, true>, k_gen2_part<false, true, true>,
                                            k_gen2_part<true, false, true>,  k_gen2_part<true, true, true>};
const GenPartKernel GENERATE_PART_KERNELS[4] = {k_generate_part<false, SD_L_MAX>, k_generate_part<true, SD_L_MAX>,
                                                k_generate_part<false, 32>, k_generate_part<true, 32>};
constexpr size_t GENERATE_PART_SMEM64 = ((sizeof(GenSharedT<SD_L_MAX>) + 15) & ~(size_t)15) + sizeof(GenPartStage);
constexpr size_t GENERATE_PART_SMEM32 = ((sizeof(GenSharedT<32>) + 15) & ~(size_t)15) + sizeof(GenPartStage);

}  // namespace

// ---------------------------------------------------------------------------------------------
// Per-device state of this translation unit: the __constant__ hash / binomial tables and the dynamic shared-memory
// limits of the generator kernels.  Constants and function attributes belong to the CURRENT device, so this runs for
// every context (symdel_create, under its lock) — never behind a process-wide flag.
cudaError_t sd_generate_setup() {
    u64 R[32], Bpow[SD_L_MAX + 1], Binv[SD_D_MAX + 1];
    u64 st = 0x243f6a8885a308d3ull;
    for (int c = 0; c < 32; ++c) R[c] = splitmix64(st) | 1ull;
    const u64 B = splitmix64(st) | 1ull;
    Bpow[0] = 1;
    for (int j = 1; j <= SD_L_MAX; ++j) Bpow[j] = Bpow[j - 1] * B;
    u64 inv = B;  // Newton iteration for the inverse modulo 2^64
    for (int it = 0; it < 6; ++it) inv *= 2 - B * inv;
    Binv[0] = 1;
    for (int m = 1; m <= SD_D_MAX; ++m) Binv[m] = Binv[m - 1] * inv;
    u32 binom[(SD_L_MAX + 1) * (SD_D_MAX + 1)], vcum[(SD_L_MAX + 1) * (SD_D_MAX + 2)];
    for (int n = 0; n <= SD_L_MAX; ++n) {
        for (int k = 0; k <= SD_D_MAX; ++k) {
            u64 c = 1;
            if (k > n) c = 0;
            else
                for (int t = 1; t <= k; ++t) c = c * (u64)(n - k + t) / (u64)t;
            binom[n * (SD_D_MAX + 1) + k] = (u32)c;
        }
        u32 acc = 0;
        for (int k = 0; k <= SD_D_MAX + 1; ++k) {
            vcum[n * (SD_D_MAX + 2) + k] = acc;
            if (k <= SD_D_MAX) acc += binom[n * (SD_D_MAX + 1) + k];
        }
    }
    cudaError_t e;
    if ((e = cudaMemcpyToSymbol(c_R, R, sizeof(R))) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbol(c_Bpow, Bpow, sizeof(Bpow))) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbol(c_Binv, Binv, sizeof(Binv))) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbol(c_binom, binom, sizeof(binom))) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbol(c_vcum, vcum, sizeof(vcum))) != cudaSuccess) return e;
    const int gsm = (int)(sizeof(GenShared) + 8 * 256 * 4);
    if ((e = cudaFuncSetAttribute(k_generate<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, gsm)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_generate<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, gsm)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_generate<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, gsm)) != cudaSuccess) return e;
    for (GenPartKernel k : GEN2_PART_KERNELS)
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GenPartShared))) != cudaSuccess) return e;
    for (int i = 0; i < 4; ++i)
        if ((e = cudaFuncSetAttribute(GENERATE_PART_KERNELS[i], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)(i < 2 ? GENERATE_PART_SMEM64 : GENERATE_PART_SMEM32))) != cudaSuccess) return e;
    return cudaSuccess;
}

cudaError_t sd_prepare(SeqSetDev s, int d, int is_b, int prefix, DevInfo* info, cudaStream_t st, i64* launches) {
    if (s.n == 0) return cudaSuccess;
    int blocks = (int)std::min<i64>((s.n + 255) / 256, 148 * 8);
    k_prepare<<<blocks, 256, 0, st>>>(s, d, is_b, prefix > 0 ? prefix : SD_L_MAX, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_check_residues(SeqSetDev s, DevInfo* info, cudaStream_t st) {
    if (s.n == 0) return cudaSuccess;
    k_check_residues<<<(int)std::min<i64>((s.n + 15) / 16, 148 * 8), 256, 0, st>>>(s, info);
    return cudaGetLastError();
}

cudaError_t sd_count(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, u32* cnt, DevInfo* info, cudaStream_t st,
                     i64* launches) {
    const bool fast = use_fast(lay, width);
    GenParams P = fast ? make_params2(a, b, lay, width) : make_params(a, b, lay, width);
    if (P.groups_total == 0) return cudaSuccess;
    P.cnt = cnt;
    P.info = info;
    if (fast) gen2_pick<true>(lay.n_chunks > 1, 0)<<<gen2_grid(P.groups_total), G2_THREADS, sizeof(Gen2Shared), st>>>(P);
    else if (lay.n_chunks > 1) k_generate<true, true><<<gen_grid(P.groups_total), GEN_THREADS, sizeof(GenShared), st>>>(P);
    else k_count_dp<<<(unsigned)((a.n + b.n + 127) / 128), 128, 0, st>>>(a, b, lay.d, lay.thinning, (int)P.prefix, cnt);
    if (launches) ++*launches;
    return cudaGetLastError();
}

i64 sd_scan_tiles(i64 n) { return (n + SC_TILE - 1) / SC_TILE; }

cudaError_t sd_scan_counts(const u32* cnt, i64 n, u64* rec_off, u64* lb_status, DevInfo* info, cudaStream_t st,
                           i64* launches) {
    const i64 tiles = std::max<i64>(1, sd_scan_tiles(n));
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    k_scan_counts<<<(unsigned)tiles, SC_THREADS, 0, st>>>(cnt, n, rec_off, lb_status, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_generate(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, const u64* rec_off, u64* records,
                        u32* ghist, int hist_bit, int npass, DevInfo* info, cudaStream_t st, i64* launches) {
    const bool fast = use_fast(lay, width);
    GenParams P = fast ? make_params2(a, b, lay, width) : make_params(a, b, lay, width);
    if (P.groups_total == 0) return cudaSuccess;
    P.rec_off = rec_off;
    P.records = records;
    P.ghist = ghist;
    P.npass = npass;
    P.hshift = hist_bit - lay.id_bits;
    P.info = info;
    if (fast)
        gen2_pick<false>(lay.n_chunks > 1, npass)<<<gen2_grid(P.groups_total), G2_THREADS,
                                                      sizeof(Gen2Shared) + (size_t)npass * 256 * 4, st>>>(P);
    else if (lay.n_chunks > 1)
        k_generate<false, true><<<gen_grid(P.groups_total), GEN_THREADS, sizeof(GenShared) + (size_t)npass * 256 * 4, st>>>(P);
    else
        k_generate<false, false><<<gen_grid(P.groups_total), GEN_THREADS, sizeof(GenShared) + (size_t)npass * 256 * 4, st>>>(P);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// Fused generation + level-1 partition (fast generator only: see sd_gen_part_applies).  bins: 256 x cap1
// records; cur: 256 cursors, zeroed here.  info->part_overflow != 0 afterwards: a bin was full.
bool sd_gen_part_applies(const Layout& lay, int width) {
    (void)width;
    return lay.hash_bits >= 8;
}

bool sd_gen_part_sliceable(const Layout& lay, int width) { return use_fast_part(lay, width); }

cudaError_t sd_gen_part(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, u64* bins, u32* cur, u64 cap1,
                        double records_per_residue, double avg_len, i64 task_begin, i64 task_end, int cursors_cleared, DevInfo* info,
                        cudaStream_t st, i64* launches) {
    // task_end == -2 / -3: set A only / set B only (cross-search with the query filter: the queries are generated first)
    const int which = task_end == -2 ? 1 : task_end == -3 ? 2 : 0;
    if (which) task_end = -1;
    const bool fast = use_fast_part(lay, width);
    GenPartParams PP{};
    PP.g = fast ? make_params2(a, b, lay, width) : make_params(a, b, lay, width);
    if (PP.g.groups_total == 0) return cudaSuccess;
    PP.g.info = info;
    PP.bins = bins;
    PP.cur = cur;
    PP.cap1 = (u32)cap1;
    {   // a batch fills the 32 lanes with residues: about 32 * records_per_residue records (thinning and padding: ~0.85)
        // d = 3: the unit of a round is a step of GP_TRIP triple iterations (about 0.55 of the lane slots make a record)
        (void)avg_len;
        const double per_round = lay.d == 3 ? GP_NW * 32.0 * GP_TRIP * 0.55 : GP_NW * 32.0 * std::max(records_per_residue, 0.03) * 0.85;
        PP.batches = (u32)std::min(8.0, std::max(1.0, std::floor(GP_ROUND / per_round + 0.5)));
    }
    // Warp tasks of k_gen2_part: every warp should get many — the last task of the slowest warp of a block keeps the other
    // seven waiting at the round barriers.  With 32-sequence tasks config 5 (d = 3, ~740 records per sequence) had 1.7 tasks per
    // warp and spent 43 % of its warp time at the round barrier: tasks of 2 sequences 1.90 -> 1.41 ms.  At d <= 2 a smaller task
    // costs more than it balances (every task end breaks the packing of sequences into lanes: config 3 with 16: +2 %), so
    // tasks shrink only below 8 per warp.
    PP.task_seqs = 32;
    if (fast) {
        const i64 warps = (i64)148 * GP_MINB * GP_NW;
        const i64 want = lay.d == 3 ? 64 : 8, low = lay.d == 3 ? 2 : 4;
        const i64 n_launch = which == 1 ? a.n : which == 2 ? b.n : task_end >= 0 ? std::min<i64>(a.n + b.n, (task_end - task_begin) * 32) : a.n + b.n;  // (what THIS launch covers)
        while (PP.task_seqs > low && n_launch / PP.task_seqs < want * warps) PP.task_seqs >>= 1;
        PP.g.groups_a = (a.n + PP.task_seqs - 1) / PP.task_seqs;
        PP.g.groups_total = PP.g.groups_a + (b.n + PP.task_seqs - 1) / PP.task_seqs;
    }
    // task range of this launch, given in units of 32 sequences: [task_begin, task_end); (0, -1) = all.  Only the launch that
    // starts at task 0 clears the cursors.
    const bool sliced = task_end >= 0;
    const i64 per32 = 32 / PP.task_seqs;
    PP.task_begin = sliced ? task_begin * per32 : 0;
    PP.task_end = sliced ? std::min(task_end * per32, PP.g.groups_total) : PP.g.groups_total;
    if (sliced && (!fast || b.n != 0)) return cudaErrorInvalidValue;  // (slices are ranges of set A: self-search)
    if (which && !fast) return cudaErrorInvalidValue;
    if (which == 1) PP.task_end = PP.g.groups_a;
    if (which == 2) PP.task_begin = PP.g.groups_a;
    if (PP.task_begin >= PP.task_end && PP.task_begin > 0) return cudaSuccess;
    cudaError_t e;
    if (PP.task_begin == 0 && !cursors_cleared && (e = cudaMemsetAsync(cur, 0, 256 * sizeof(u32), st)) != cudaSuccess) return e;
    if (fast) {
        const int grid = (int)std::min<i64>((PP.task_end - PP.task_begin + GP_NW - 1) / GP_NW, 148 * GP_MINB);
        const bool plain = lay.hash_bits + lay.id_bits == 64 && lay.id_bits <= 31;
        GEN2_PART_KERNELS[(lay.d == 3 ? 4 : 0) + (lay.n_chunks > 1 ? 2 : 0) + (plain ? 1 : 0)]<<<grid, GP_THREADS, sizeof(GenPartShared), st>>>(PP);
    } else {
        const bool narrow = width - 1 <= 32;  // rows of 32 residues: a fourth block fits on the SM
        const int grid = (int)std::min<i64>(PP.g.groups_total, 148 * (narrow ? GQ_MINB + 1 : GQ_MINB));
        GENERATE_PART_KERNELS[(narrow ? 2 : 0) + (lay.n_chunks > 1 ? 1 : 0)]<<<grid, GEN_THREADS, narrow ? GENERATE_PART_SMEM32 : GENERATE_PART_SMEM64, st>>>(PP);
    }
    if (launches) ++*launches;
    return cudaGetLastError();
}
