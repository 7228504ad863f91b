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
// per text character it costs ~15 bit operations instead of a column of min/add.  Sequences are
// pre-packed (k_pack) into five bit-planes of their 5-bit residue codes; the match mask Eq[c] is
// rebuilt from the pattern's and the text's planes rather than looked up in a 32-entry table, which
// keeps the whole state in registers and makes each sequence one aligned 32/48-byte gather.
// Survivors are compacted in order (block scan + decoupled look-back), so the output stays sorted.
#include "kernels.h"

namespace {

// ---- packed sequences: five bit-planes of the 5-bit residue codes + the length ---------------------
// plane k, bit j = bit k of residue j.  NARROW (longest sequence <= 32): 8 x u32 = 32 B per sequence
// {b0, b1, b2, b3, b4, len, 0, 0}; WIDE: 6 x u64 = 48 B {b0 .. b4, len}.  One aligned 32/48-byte gather
// per sequence replaces two offset loads and ~15 unaligned byte loads in the verifier.
template <typename W>
struct Planes {
    W b[5];
    int len;
};

template <typename W>
__device__ __forceinline__ Planes<W> load_planes(const void* slots, u64 id);
template <>
__device__ __forceinline__ Planes<u32> load_planes<u32>(const void* slots, u64 id) {
    const uint4* p = reinterpret_cast<const uint4*>(slots) + 2 * id;
    const uint4 lo = __ldg(p), hi = __ldg(p + 1);
    Planes<u32> r;
    r.b[0] = lo.x, r.b[1] = lo.y, r.b[2] = lo.z, r.b[3] = lo.w, r.b[4] = hi.x;
    r.len = (int)hi.y;
    return r;
}
template <>
__device__ __forceinline__ Planes<u64> load_planes<u64>(const void* slots, u64 id) {
    const ulonglong2* p = reinterpret_cast<const ulonglong2*>(slots) + 3 * id;
    const ulonglong2 x = __ldg(p), y = __ldg(p + 1), z = __ldg(p + 2);
    Planes<u64> r;
    r.b[0] = x.x, r.b[1] = x.y, r.b[2] = y.x, r.b[3] = y.y, r.b[4] = z.x;
    r.len = (int)z.y;
    return r;
}

template <typename W>
__global__ void __launch_bounds__(256) k_pack(SeqSetDev A, SeqSetDev B, void* slots, DevInfo* info) {
    const i64 g = (i64)blockIdx.x * 256 + threadIdx.x;
    if (g >= A.n + B.n) return;
    const SeqSetDev& S = g < A.n ? A : B;
    const i64 i = g < A.n ? g : g - A.n;
    const i64 o = S.off[i];
    const int L = (int)(S.off[i + 1] - o);
    W b[5] = {0, 0, 0, 0, 0};
    bool bad = false;
    for (int j = 0; j < L; ++j) {
        const W c = (W)(unsigned char)S.seqs[o + j];
        bad |= c < 1 || c > 31;  // S0: residue codes 1..31 (0 is reserved)
#pragma unroll
        for (int k = 0; k < 5; ++k) b[k] |= ((c >> k) & 1) << j;
    }
    if (bad) atomicOr(&info->err, (u32)SD_ERR_RESIDUE);
    if (sizeof(W) == 4) {
        uint4* p = reinterpret_cast<uint4*>(slots) + 2 * g;
        p[0] = make_uint4((u32)b[0], (u32)b[1], (u32)b[2], (u32)b[3]);
        p[1] = make_uint4((u32)b[4], (u32)L, 0u, 0u);
    } else {
        ulonglong2* p = reinterpret_cast<ulonglong2*>(slots) + 3 * g;
        p[0] = make_ulonglong2(b[0], b[1]);
        p[1] = make_ulonglong2(b[2], b[3]);
        p[2] = make_ulonglong2(b[4], (u64)L);
    }
}

// Bit-parallel global edit distance (Myers 1999 / Hyyro 2003).  Pattern and text both arrive as
// bit-planes; the match mask of text character i is Eq = AND_k ~(P_k xor -(T_k >> i & 1)).
template <typename W>
__device__ __forceinline__ int myers_lev(const Planes<W>& P, const Planes<W>& T) {
    const int m = P.len, n = T.len;
    if (m == 0) return n;
    if (n == 0) return m;
    const W mask = (m == (int)(8 * sizeof(W))) ? ~(W)0 : (((W)1 << m) - 1);
    const W top = (W)1 << (m - 1);
    W Pv = mask, Mv = 0;
    int score = m;
    for (int i = 0; i < n; ++i) {
        W Eq = mask;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const W mk = (W)0 - ((T.b[k] >> i) & 1);
            Eq &= ~(P.b[k] ^ mk);
        }
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

// Hamming mode (NEXT-3, Fig. S3): defined for equal lengths only; a position differs iff any of
// the five code bit-planes differs.  Returns > any threshold for unequal lengths.
template <typename W>
__device__ __forceinline__ int hamming_planes(const Planes<W>& P, const Planes<W>& T) {
    if (P.len != T.len) return 1 << 20;
    W x = 0;
#pragma unroll
    for (int k = 0; k < 5; ++k) x |= P.b[k] ^ T.b[k];
    return sizeof(W) == 8 ? __popcll((unsigned long long)x) : __popc((unsigned)x);
}

constexpr int VF_THREADS = 256;
// candidates per thread: 8 when most candidates are repeats (unfiltered: 4 per thread 0.087 -> 8: 0.077 ms on config 3),
// 2 when the duplicate filter ran first (nearly every candidate then needs a distance: small tiles spread them over the SMs)
constexpr int VF_IPT_RAW = 8, VF_IPT_FILTERED = 2;

// Tile of VF_TILE = 2048 sorted candidates: (1) flag the unique ones and compact their positions into shared
// memory, (2) spread the COMPACTED list over the threads for the distance computation (after dedup
// only a fraction of the candidates is left: this keeps every lane busy), (3) ordered compaction of
// the survivors (block scan + 32-wide decoupled look-back) so the output stays sorted.
// DIRECT: this call is known to be the only flush of the whole search, so the survivors are final: they are
// unpacked straight into (out_i, out_j, out_dist) (first surv_capacity of them) and info->n_out = their number.
template <typename W, bool DIRECT, int VF_IPT>
__global__ void __launch_bounds__(VF_THREADS) k_verify(const u64* __restrict__ cand, u64 n, const u64* __restrict__ n_dev,
                                                      const void* __restrict__ slots,
                                                      Layout lay, u64* __restrict__ surv, u64 surv_base,
                                                      u64 surv_capacity, u64* lb_status, DevInfo* info,
                                                      i32* __restrict__ out_i, i32* __restrict__ out_j,
                                                      i32* __restrict__ out_dist) {
    constexpr int VF_TILE = VF_THREADS * VF_IPT;
    __shared__ unsigned short s_list[VF_TILE];
    __shared__ unsigned char s_res[VF_TILE];
    __shared__ u32 s_warp[VF_THREADS / 32 + 1];
    __shared__ u32 s_tile, s_nuniq;
    __shared__ u64 s_excl;
    const u32 tid = threadIdx.x, lane = tid & 31;
    if (n_dev) n = *n_dev;  // the count lives on the device; the grid was sized for an upper bound
    if (tid == 0) {
        s_tile = atomicAdd(&info->ticket[SD_TK_VERIFY], 1u);
        if (s_tile == gridDim.x - 1) info->ticket[SD_TK_VERIFY] = 0;
        s_nuniq = 0;
    }
    __syncthreads();
    const u32 tile = s_tile;
    const u64 base = (u64)tile * VF_TILE;
    const u32 last_tile = n ? (u32)((n - 1) / VF_TILE) : 0u;
    if (n == 0 && tile == 0 && tid == 0) {
        info->n_surv = surv_base;
        if (DIRECT) info->n_out = 0;
    }
    if (base >= n) return;  // surplus block (block-uniform): tiles are ticket-numbered, nobody waits on it
    const u32 tile_n = (u32)min((u64)VF_TILE, n - base);
    const u64 bmask = (1ull << lay.b_bits) - 1ull;

    // ---- (1) unique flags, compacted positions ----
#pragma unroll
    for (int k = 0; k < VF_IPT; ++k) {
        const u32 pos = k * VF_THREADS + tid;
        const u64 c = pos < tile_n ? cand[base + pos] : 0ull;
        u64 prev = __shfl_up_sync(SD_FULL, c, 1);
        if (lane == 0) prev = (pos < tile_n && base + pos > 0) ? cand[base + pos - 1] : ~c;
        bool uniq = pos < tile_n && c != prev;
        if (!lay.cross && (c >> lay.b_bits) == (c & bmask)) uniq = false;  // same sequence twice in one run
        const u32 bal = __ballot_sync(SD_FULL, uniq);
        u32 wbase = 0;
        if (lane == 0 && bal) wbase = atomicAdd(&s_nuniq, (u32)__popc(bal));
        wbase = __shfl_sync(SD_FULL, wbase, 0);
        if (uniq) s_list[wbase + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)pos;
        if (pos < VF_TILE) s_res[pos] = 0xff;
    }
    __syncthreads();
    const u32 nuniq = s_nuniq;

    // ---- (2) distances over the compacted list ----
    for (u32 e = tid; e < nuniq; e += VF_THREADS) {
        const u32 pos = s_list[e];
        const u64 c = cand[base + pos];
        const u64 a = c >> lay.b_bits, b = c & bmask;
        const Planes<W> pa = load_planes<W>(slots, a);
        const Planes<W> pb = load_planes<W>(slots, lay.cross ? (u64)lay.n_a + b : b);
        const int dl = pa.len > pb.len ? pa.len - pb.len : pb.len - pa.len;
        if (dl <= lay.d) {
            const int dist = lay.metric ? hamming_planes<W>(pa, pb) : myers_lev<W>(pa, pb);
            if (dist <= lay.d) s_res[pos] = (unsigned char)dist;
        }
    }
    __syncthreads();

    // ---- (3) ordered compaction (thread owns VF_IPT consecutive positions) ----
    u32 keepmask = 0, cntk = 0;
#pragma unroll
    for (int k = 0; k < VF_IPT; ++k) {
        const u32 pos = tid * VF_IPT + k;
        if (s_res[pos] != 0xff) keepmask |= 1u << k, ++cntk;
    }
    u32 total;
    const u32 rank = sd_block_excl_sum<VF_THREADS>(cntk, &total, s_warp);
    if (tid < 32) {
        const u64 excl = sd_lookback_warp(lb_status, tile, total);
        if (tid == 0) {
            s_excl = excl;
            if (nuniq) atomicAdd((unsigned long long*)&info->n_unique, (unsigned long long)nuniq);
            if (tile == last_tile) {
                info->n_surv = surv_base + excl + total;
                if (DIRECT) info->n_out = excl + total;
            }
        }
    }
    __syncthreads();
    u64 out = surv_base + s_excl + rank;
#pragma unroll
    for (int k = 0; k < VF_IPT; ++k) {
        if (keepmask & (1u << k)) {
            const u32 pos = tid * VF_IPT + k;
            if (DIRECT) {
                if (out < surv_capacity) {  // beyond the caller's capacity: counted, not written (SYMDEL_E_CAPACITY)
                    const u64 c = cand[base + pos];
                    out_i[out] = (i32)(c >> lay.b_bits);
                    out_j[out] = (i32)(c & bmask);
                    out_dist[out] = (i32)s_res[pos];
                }
            } else if (out < surv_capacity) {
                surv[out] = (cand[base + pos] << 3) | (u64)s_res[pos];
            } else {
                info->surv_overflow = 1u;
            }
            ++out;
        }
    }
}

constexpr int FN_THREADS = 256;

// packed_out != nullptr: the kept survivors are written back as packed words (the survivor-list merge between
// flushes) instead of being unpacked to the SoA outputs.
__global__ void __launch_bounds__(FN_THREADS) k_finalize(const u64* __restrict__ surv, u64 n, Layout lay, int dedup,
                                                        i32* __restrict__ out_i, i32* __restrict__ out_j,
                                                        i32* __restrict__ out_dist, u64* __restrict__ packed_out,
                                                        u64 capacity, u64* lb_status, DevInfo* info) {
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
        if (packed_out) {
            if (pos < capacity) packed_out[pos] = v;
        } else if (pos < capacity) {
            const u64 pr = v >> 3;
            out_i[pos] = (i32)(pr >> lay.b_bits);
            out_j[pos] = (i32)(pr & ((1ull << lay.b_bits) - 1ull));
            out_dist[pos] = (i32)(v & 7ull);
        }
    }
}

template <typename W>
__global__ void __launch_bounds__(256) k_lev_pairs(const void* __restrict__ slots, i64 n_a, i64 n_b, const i32* __restrict__ ia,
                                                   const i32* __restrict__ ib, i64 n, i32* __restrict__ dist, u32* err) {
    const i64 t = (i64)blockIdx.x * 256 + threadIdx.x;
    if (t >= n) return;
    const i64 a = ia[t], b = ib[t];
    if (a < 0 || a >= n_a || b < 0 || b >= n_b) {  // caller-supplied indices: never gather out of bounds
        dist[t] = -1;
        atomicOr(err, (u32)SD_ERR_INTERNAL);
        return;
    }
    dist[t] = myers_lev<W>(load_planes<W>(slots, (u64)a), load_planes<W>(slots, (u64)(n_a + b)));
}

// ---- NEXT-4: M x M repertoire-overlap matrix --------------------------------------------
// "a wrapper that aggregates an M x M overlap matrix from identified neighbor pairs, where each entry
// contains the number of neighbors between two repertoires".  One pass over the output pairs: block-private
// shared-memory histogram (M <= 64), flushed with one 64-bit global atomic per non-zero cell.
constexpr int OV_THREADS = 256, OV_MMAX_SMEM = 64;

__global__ void __launch_bounds__(OV_THREADS) k_overlap(const i32* __restrict__ pi, const i32* __restrict__ pj, u64 n,
                                                       const i32* __restrict__ lab_i, i64 n_i, const i32* __restrict__ lab_j,
                                                       i64 n_j, int M, int symmetric, unsigned long long* __restrict__ matrix,
                                                       u32* err) {
    extern __shared__ u32 s_cell[];
    const bool use_smem = M <= OV_MMAX_SMEM;
    if (use_smem) {
        for (int c = threadIdx.x; c < M * M; c += OV_THREADS) s_cell[c] = 0;
        __syncthreads();
    }
    const u64 stride = (u64)gridDim.x * OV_THREADS;
    for (u64 t = (u64)blockIdx.x * OV_THREADS + threadIdx.x; t < n; t += stride) {
        const i64 xi = pi[t], xj = pj[t];
        if (xi < 0 || xi >= n_i || xj < 0 || xj >= n_j) {  // a pair index outside its label array
            atomicOr(err, (u32)SD_ERR_INTERNAL);
            continue;
        }
        const i32 a = lab_i[xi], b = lab_j[xj];
        if (a < 0 || a >= M || b < 0 || b >= M) {
            atomicOr(err, (u32)SD_ERR_INTERNAL);
            continue;
        }
        if (use_smem) {
            atomicAdd(&s_cell[a * M + b], 1u);
            if (symmetric && a != b) atomicAdd(&s_cell[b * M + a], 1u);
        } else {
            atomicAdd(&matrix[(u64)a * M + b], 1ull);
            if (symmetric && a != b) atomicAdd(&matrix[(u64)b * M + a], 1ull);
        }
    }
    if (use_smem) {
        __syncthreads();
        for (int c = threadIdx.x; c < M * M; c += OV_THREADS)
            if (s_cell[c]) atomicAdd(&matrix[c], (unsigned long long)s_cell[c]);
    }
}

}  // namespace

// matrix (M x M, row-major, zeroed here) += the label pairs of the n output pairs; *err gets SD_ERR_INTERNAL if
// a label lies outside [0, M)
cudaError_t sd_overlap(const i32* pi, const i32* pj, i64 n, const i32* lab_i, i64 n_i, const i32* lab_j, i64 n_j, int M,
                       int symmetric, u64* matrix, u32* err, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(matrix, 0, (size_t)M * M * 8, st);
    if (e != cudaSuccess || n == 0) return e;
    const unsigned blocks = (unsigned)std::min<i64>((n + OV_THREADS * 8 - 1) / (OV_THREADS * 8), 148 * 8);
    const size_t smem = M <= OV_MMAX_SMEM ? (size_t)M * M * 4 : 0;
    k_overlap<<<blocks, OV_THREADS, smem, st>>>(pi, pj, (u64)n, lab_i, n_i, lab_j, n_j, M, symmetric, (unsigned long long*)matrix, err);
    return cudaGetLastError();
}

i64 sd_verify_tiles(i64 n) { return (n + VF_THREADS * VF_IPT_FILTERED - 1) / (VF_THREADS * VF_IPT_FILTERED); }  // (the smaller tile: sizes lb_status)

i64 sd_pack_bytes(i64 n_total, int maxlen) { return n_total * (maxlen <= 32 ? 32 : 48); }

cudaError_t sd_pack(SeqSetDev a, SeqSetDev b, int maxlen, void* slots, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 n = a.n + b.n;
    if (n == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (maxlen <= 32) k_pack<u32><<<blocks, 256, 0, st>>>(a, b, slots, info);
    else k_pack<u64><<<blocks, 256, 0, st>>>(a, b, slots, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// filtered candidates (n_dev set) take the small tile
template <typename W, bool DIRECT, typename... Args>
static void vf_launch(bool filtered, i64 tiles, cudaStream_t st, Args... args) {
    if (filtered) k_verify<W, DIRECT, VF_IPT_FILTERED><<<(unsigned)tiles, VF_THREADS, 0, st>>>(args...);
    else k_verify<W, DIRECT, VF_IPT_RAW><<<(unsigned)tiles, VF_THREADS, 0, st>>>(args...);
}
static i64 vf_tiles(i64 n, bool filtered) {
    const i64 t = VF_THREADS * (filtered ? VF_IPT_FILTERED : VF_IPT_RAW);
    return (n + t - 1) / t;
}

cudaError_t sd_verify(const u64* cand, i64 n_cand, const u64* n_dev, const void* slots, const Layout& lay, int maxlen, u64* surv,
                      u64 surv_base, u64 surv_capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = vf_tiles(n_cand, n_dev != nullptr);
    if (tiles == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    if (maxlen <= 32)
        vf_launch<u32, false>(n_dev != nullptr, tiles, st, cand, (u64)n_cand, n_dev, slots, lay, surv, surv_base, surv_capacity,
                                                                     lb_status, info, (i32*)nullptr, (i32*)nullptr, (i32*)nullptr);
    else
        vf_launch<u64, false>(n_dev != nullptr, tiles, st, cand, (u64)n_cand, n_dev, slots, lay, surv, surv_base, surv_capacity,
                                                                     lb_status, info, (i32*)nullptr, (i32*)nullptr, (i32*)nullptr);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// The only flush of a search: unique + verify + unpack in one kernel.  info->n_out = number of result pairs
// (the first `capacity` are written).
cudaError_t sd_verify_direct(const u64* cand, i64 n_cand, const u64* n_dev, const void* slots, const Layout& lay, int maxlen, i32* out_i,
                             i32* out_j, i32* out_dist, i64 capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = vf_tiles(n_cand, n_dev != nullptr);
    if (tiles == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    if (maxlen <= 32)
        vf_launch<u32, true>(n_dev != nullptr, tiles, st, cand, (u64)n_cand, n_dev, slots, lay, (u64*)nullptr, (u64)0, (u64)capacity, lb_status,
                                                                    info, out_i, out_j, out_dist);
    else
        vf_launch<u64, true>(n_dev != nullptr, tiles, st, cand, (u64)n_cand, n_dev, slots, lay, (u64*)nullptr, (u64)0, (u64)capacity, lb_status,
                                                                    info, out_i, out_j, out_dist);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t sd_finalize(const u64* surv, i64 n_surv, const Layout& lay, int dedup, i32* out_i, i32* out_j, i32* out_dist,
                        u64* packed_out, i64 capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches) {
    const i64 tiles = (n_surv + FN_THREADS - 1) / FN_THREADS;
    if (tiles == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lb_status, 0, (size_t)tiles * 8, st);
    if (e != cudaSuccess) return e;
    k_finalize<<<(unsigned)tiles, FN_THREADS, 0, st>>>(surv, (u64)n_surv, lay, dedup, out_i, out_j, out_dist, packed_out,
                                                       (u64)capacity, lb_status, info);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// distances for index pairs (stage test): slots hold set A followed by set B
cudaError_t sd_lev_pairs(const void* slots, i64 n_a, i64 n_b, int maxlen, const i32* ia, const i32* ib, i64 n_pairs, i32* dist,
                         u32* err, cudaStream_t st) {
    if (n_pairs == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n_pairs + 255) / 256);
    if (maxlen <= 32) k_lev_pairs<u32><<<blocks, 256, 0, st>>>(slots, n_a, n_b, ia, ib, n_pairs, dist, err);
    else k_lev_pairs<u64><<<blocks, 256, 0, st>>>(slots, n_a, n_b, ia, ib, n_pairs, dist, err);
    return cudaGetLastError();
}
