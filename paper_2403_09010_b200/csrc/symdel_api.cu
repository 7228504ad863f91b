// symdel_api.cu — the C ABI of include/symdel.h and the host-side pipeline (S0-S5).
//
// One call (App. F.3 "XTNeighbor base algorithm", re-designed):
//   S0  prepare : validate CSR input, longest sequence, upper bound of the record count, pack for the verifier
//   for each key-range chunk c of P (S5; P = 1 when the workspace allows), one of two pipelines:
//     FUSED (default)                                        EXACT (options, or after an overflow)
//     S1+S2 k_gen*_part : variants hashed and staged under   S1 count + scan + generate : records in id order
//           their top 8 hash bits -> 256 fixed-capacity bins S2 onesweep passes on exact histograms (8 bits each)
//     S2    k_part2     : next b2 bits -> fixed-capacity     S3a k_join_fast (one window) else k_join (windowed,
//           buckets with counts                                  chunks oversized buckets)
//     S3a   k_join_bkt  : shared-memory hash join per bucket
//     then, per window of the candidate buffer:
//       S3b sort the packed pair ids; S4 unique + verify -> survivors (pair << 3 | dist) appended in order,
//           or straight into the outputs when the window is the only flush of the search
//   if more than one flush happened: sort survivors, unique, unpack -> (out_i, out_j, out_dist), ascending (i, j)
// Equal keys always land in the same chunk and a verified pair carries the same distance wherever it
// was found, so chunking and windowing change memory use only.  This replaces the paper's 2-D-buffer
// streaming (App. C; App. F.4) whose purpose — bounded memory — it serves.
//
// Host <-> device crossings per call (fused, one chunk, one window): one pinned-memory read-back after S0,
// one after the join (candidate count, overflow flags), one at the end.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/symdel.h"
#include "kernels.h"

struct symdel_ctx {
    int device = 0;
    cudaError_t last_cuda = cudaSuccess;
    symdel_stats stats{};
    int opt_timing = 0;
    i64 opt_force_chunks = 0, opt_cand_cap = 0, opt_hash_bits = 0, opt_no_thinning = 0, opt_general_gen = 0;
    i64 opt_sort_variant = 0, opt_surv_cap = 0, opt_cand_filter = 0, opt_no_query_filter = 0, opt_flush_per_chunk = 0;
    i64 opt_sort_bits = -1, opt_sort_stable = 0, opt_sort_grouping = 0, opt_join_general = 0, opt_exact = 0, opt_prefix = 0, opt_metric = 0;
    DevInfo* h_info = nullptr;  // pinned; followed by 256 u32 (the level-1 bin counts of the fused pipeline)
    void* arena = nullptr;      // device arena of the *_host entry points: outputs + workspace
    size_t arena_bytes = 0;
    void* in_arena = nullptr;   // ... and their inputs (separate: the copies start before the workspace size is known)
    size_t in_arena_bytes = 0;
    cudaStream_t stream = nullptr;  // stream of the *_host entry points
    cudaStream_t side = nullptr;    // the verifier's bit-plane table is packed here, beside generation (forked from / joined into the caller's stream by events)
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bool side_pending = false;      // work was forked to `side` and the caller's stream has not been made to wait for it yet
    std::vector<cudaEvent_t> events;
    std::vector<cudaEvent_t> hp_events;  // host entry points: arrival of the input slices
};

namespace {

#define CK(call)                                  \
    do {                                          \
        cudaError_t e__ = (call);                 \
        if (e__ != cudaSuccess) {                 \
            ctx->last_cuda = e__;                 \
            return SYMDEL_E_CUDA;                 \
        }                                         \
    } while (0)

inline i64 align_up(i64 x, i64 a = 256) { return (x + a - 1) / a * a; }

struct Bump {
    char* base;
    i64 size, used = 0;
    bool ok = true;
    Bump(void* p, i64 n) : base((char*)p), size(n) {}
    template <typename T>
    T* take(i64 count) {
        i64 bytes = align_up(count * (i64)sizeof(T));
        if (used + bytes > size) {
            ok = false;
            return nullptr;
        }
        T* r = (T*)(base + used);
        used += bytes;
        return r;
    }
    i64 left() const { return size - used; }
};

int bits_for(i64 count) {  // smallest b >= 1 with 2^b >= count (values 0 .. count-1 fit)
    int b = 1;
    while (((i64)1 << b) < count) ++b;
    return b;
}

u64 vcount_host(int L, int d) {
    u64 acc = 0, c = 1;
    for (int k = 0; k <= d; ++k) {
        if (k > L) break;
        if (k > 0) c = c * (u64)(L - k + 1) / (u64)k;
        acc += c;
    }
    return acc;
}

// Fused pipeline (generation + level-1 partition, level-2 partition, bucket join): fixed-capacity bins
// and buckets sized for `nexp` expected records with hash-uniform keys, + 8 standard deviations.
struct FusedPlan {
    int b, b2;        // partitioned hash bits in all (12..16) and at level 2
    i64 cap1, cap2;   // records per level-1 bin / level-2 bucket (multiples of 32)
    i64 bins_rec, bkt_rec, nbuckets;
};
constexpr i64 FUSED_MAX_BUCKETS = 65536;
FusedPlan plan_fused(i64 nexp) {
    FusedPlan f{};
    nexp = std::max<i64>(nexp, 1);
    f.b = 12;  // at least 4096 buckets: the bucket join keeps its chain links in the top 12 bits of the staged records
    while (f.b < 16 && (double)nexp / std::pow(2.0, f.b) > 1800.0) ++f.b;
    f.b2 = f.b - 8;
    auto cap_of = [](double avg) { return (i64)((avg + 8.0 * std::sqrt(avg) + 64.0 + 31.0) / 32.0) * 32; };
    f.cap1 = cap_of((double)nexp / 256.0);
    f.nbuckets = (i64)256 << f.b2;
    f.cap2 = f.b2 ? cap_of((double)nexp / (double)f.nbuckets) : 0;
    f.bins_rec = 256 * f.cap1;
    f.bkt_rec = f.b2 ? f.nbuckets * f.cap2 : 0;
    return f;
}

i64 rec_bytes(i64 ncap, int npass) {
    const FusedPlan f = plan_fused(ncap);
    return align_up(std::max(ncap, f.bins_rec) * 8) + align_up(std::max(ncap, f.bkt_rec) * 8) +
           align_up(sd_sort_scratch_bytes(ncap, npass)) + align_up((2 * sd_join_tiles(ncap) + 2) * 8);
}
i64 cand_bytes(i64 ccap, int ppass) {
    return 2 * align_up(ccap * 8) + align_up(sd_sort_scratch_bytes(ccap, ppass)) + align_up((ccap / 256 + 2) * 8);
}
i64 fixed_bytes(i64 n_total) {
    return align_up((i64)sizeof(DevInfo)) + align_up(n_total * 4) + align_up((n_total + 1) * 8) +
           align_up((sd_scan_tiles(n_total) + 1) * 8) + align_up(n_total * 48) + align_up((256 + 2 * FUSED_MAX_BUCKETS) * 4) + 4096;
}

struct Timer {
    symdel_ctx* ctx;
    cudaStream_t st;
    bool on;
    size_t next = 0;
    struct Span { int stage; size_t a, b; };
    std::vector<Span> spans;  // evaluated after the final synchronize (events must have completed)
    Timer(symdel_ctx* c, cudaStream_t s) : ctx(c), st(s), on(c->opt_timing != 0) {}
    void span(int stage, size_t a, size_t b) { if (on) spans.push_back({stage, a, b}); }
    float total(int stage) {
        float t = 0;
        for (auto& sp : spans) if (sp.stage == stage) t += ms(sp.a, sp.b);
        return t;
    }
    size_t mark() {
        if (!on) return 0;
        if (next >= ctx->events.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            ctx->events.push_back(e);
        }
        cudaEventRecord(ctx->events[next], st);
        return next++;
    }
    float ms(size_t a, size_t b) {
        float m = 0;
        if (on) cudaEventElapsedTime(&m, ctx->events[a], ctx->events[b]);
        return m;
    }
};

// The *_host entry points send the input in pieces on the side stream: all offsets first (S0 needs nothing else), then the
// residues slice by slice, so that generation starts on the first slice while the others are being copied.
constexpr int HP_MAX_SLICES = 8;
struct HostPlan {
    int n_slices = 0;                  // slices of set A's warp tasks (self-search; 1: no slicing)
    i64 task_end[HP_MAX_SLICES] = {};  // slice i = tasks [task_end[i-1], task_end[i])
    cudaEvent_t arrived[HP_MAX_SLICES] = {};
    cudaEvent_t offsets_arrived = nullptr, all_arrived = nullptr;
};

int read_info(symdel_ctx* ctx, const DevInfo* d_info, cudaStream_t st) {
    CK(cudaMemcpyAsync(ctx->h_info, d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return SYMDEL_OK;
}

int err_from_flags(u32 f) {
    if (f & SD_ERR_OFFSETS) return SYMDEL_E_OFFSETS;
    if (f & SD_ERR_TOO_LONG) return SYMDEL_E_TOO_LONG;
    if (f & SD_ERR_RESIDUE) return SYMDEL_E_RESIDUE;
    if (f & SD_ERR_INTERNAL) return SYMDEL_E_INTERNAL;
    if (f & SD_ERR_OVERFLOW) return SYMDEL_E_WORKSPACE;
    return SYMDEL_OK;
}

// -------------------------------------------------------------------------------------------------
int run_pipeline_body(symdel_ctx* ctx, SeqSetDev A, SeqSetDev B, int cross, int d, void* workspace, i64 workspace_bytes,
                 i32* out_i, i32* out_j, i32* out_dist, i64 capacity, i64* n_pairs_host, cudaStream_t st, const HostPlan* hp) {
    if (!ctx || !n_pairs_host || d < 0 || d > SD_D_MAX || A.n < 0 || B.n < 0 || capacity < 0) return SYMDEL_E_ARG;
    *n_pairs_host = 0;
    const i64 n_total = A.n + B.n;
    symdel_stats& S = ctx->stats;
    S = symdel_stats{};
    if (n_total >= ((i64)1 << 30)) return SYMDEL_E_TOO_MANY;
    if (A.n == 0 || (cross && B.n == 0)) return SYMDEL_OK;
    if (!A.seqs || !A.off || (cross && (!B.seqs || !B.off)) || !workspace) return SYMDEL_E_ARG;
    if (capacity > 0 && (!out_i || !out_j || !out_dist)) return SYMDEL_E_ARG;
    if (((uintptr_t)workspace & 255) != 0) return SYMDEL_E_ARG;
    CK(cudaSetDevice(ctx->device));
    Timer tm(ctx, st);
    const size_t ev_begin = tm.mark();

    Bump ws(workspace, workspace_bytes);
    DevInfo* info = ws.take<DevInfo>(1);
    u32* cnt = ws.take<u32>(n_total);
    u64* rec_off = ws.take<u64>(n_total + 1);
    u64* scan_lb = ws.take<u64>(sd_scan_tiles(n_total) + 1);
    if (!ws.ok) return SYMDEL_E_WORKSPACE;

    // ---- S0 ----
    CK(cudaMemsetAsync(info, 0, sizeof(DevInfo), st));
    bool info_fresh = true;  // until something other than S0 has written to the status block: the first fused attempt skips its clears
    const int prefix = (int)ctx->opt_prefix;  // App. B: exact only if the prefix is longer than the threshold
    if (prefix > 0 && prefix <= d) return SYMDEL_E_ARG;
    if (hp) CK(cudaStreamWaitEvent(st, hp->offsets_arrived, 0));  // (host entry points: S0 needs the offsets only)
    CK(sd_prepare(A, d, 0, prefix, info, st, &S.n_launches));
    if (cross) CK(sd_prepare(B, d, 1, prefix, info, st, &S.n_launches));
    int rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    const i64 nmax = (i64)ctx->h_info->nmax;
    const i64 residues = (i64)ctx->h_info->residues;
    const int maxlen = (int)ctx->h_info->maxlen;
    const size_t ev_prepared = tm.mark();
    // S5 layout: deletion sets per VARIANT length (upper bound: before thinning), cumulated.  Chunk c of P is the slice
    // [c / P, (c + 1) / P) of that axis; inside a length the slice is cut by the hash fraction (generate.cu, gen_in_chunk).
    double vl_cum[SD_L_MAX + 2];
    vl_cum[0] = 0;
    for (int vl = 0; vl <= SD_L_MAX; ++vl) {
        double w = 0;
        u64 binom = 1;  // C(vl + k, k)
        for (int k = 0; k <= d && vl + k <= SD_L_MAX; ++k) {
            if (k > 0) binom = binom * (u64)(vl + k) / (u64)k;
            w += (double)ctx->h_info->len_hist[vl + k] * (double)binom;
        }
        vl_cum[vl + 1] = vl_cum[vl] + w;
    }
    auto chunk_pos = [&](u32 c, u32 of) -> u64 {  // where chunk c of `of` starts on the (variant length << 32 | hash fraction) axis
        if (c == 0) return 0ull;
        if (c >= of) return ~0ull;
        const double target = vl_cum[SD_L_MAX + 1] * (double)c / (double)of;
        int vl = 0;
        while (vl < SD_L_MAX && vl_cum[vl + 1] <= target) ++vl;
        const double w = vl_cum[vl + 1] - vl_cum[vl];
        double frac = w > 0 ? (target - vl_cum[vl]) / w : 0;
        frac = std::min<double>(std::max<double>(frac, 0), 0.99999999);
        return ((u64)vl << 32) | (u64)(frac * 4294967296.0);
    };

    Layout lay{};
    lay.n_a = A.n;
    lay.n_b = B.n;
    lay.cross = cross;
    lay.d = d;
    lay.id_bits = bits_for(n_total + 1);
    lay.b_bits = cross ? bits_for(B.n) : lay.id_bits;
    lay.pair_bits = (cross ? bits_for(A.n) : lay.id_bits) + lay.b_bits;
    lay.thinning = ctx->opt_no_thinning ? 0 : 1;
    lay.force_general = ctx->opt_general_gen ? 1 : 0;
    lay.prefix = prefix;
    lay.metric = (int)ctx->opt_metric;
    {
        // Hash field: every bit the id leaves free (SYMDEL_OPT_HASH_BITS narrows it: more colliding
        // variants, same result).  S2 radix-partitions only its top sort_bits: enough 8-bit digits for the
        // average bucket to fit the join kernel's shared-memory window; the join compares the rest.
        const int hb_max = 64 - lay.id_bits;
        lay.hash_bits = ctx->opt_hash_bits > 0 ? (int)std::min<i64>(ctx->opt_hash_bits, hb_max) : hb_max;
    }
    // sort_bits is fixed per chunk from its actual record count; the workspace is planned for the bound
    auto pick_sort_bits = [&](i64 nrec) {
        int sb = 0;
        if (ctx->opt_sort_bits >= 0) sb = (int)ctx->opt_sort_bits;
        else
            while (sb < 56 && (double)nrec / std::pow(2.0, sb) > 1850.0) sb += 8;
        return std::min(sb, lay.hash_bits / 8 * 8);
    };
    const int npass_max = pick_sort_bits(nmax) / 8;
    const int ppass = (lay.pair_bits + 7) / 8;
    const int spass = (lay.pair_bits + 7) / 8;
    S.hash_bits = lay.hash_bits;
    S.id_bits = lay.id_bits;

    // ---- packed bit-plane table for the verifier ----
    void* slots = ws.take<char>(sd_pack_bytes(n_total, maxlen));
    u32* fcnt = ws.take<u32>(256 + 2 * FUSED_MAX_BUCKETS);  // fused pipeline: level-1 cursors | level-2 counts | redo list
    if (!ws.ok) return SYMDEL_E_WORKSPACE;
    // (only the verifier reads the table, and k_pack's residue check is looked at after the join: the kernel runs on the
    //  side stream while the caller's stream generates; join_side() makes the caller's stream wait for it)
    CK(cudaEventRecord(ctx->ev_fork, st));
    CK(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
    if (hp && hp->all_arrived) CK(cudaStreamWaitEvent(ctx->side, hp->all_arrived, 0));
    CK(sd_pack(A, B, maxlen, slots, info, ctx->side, &S.n_launches));
    CK(cudaEventRecord(ctx->ev_join, ctx->side));
    ctx->side_pending = true;
    bool input_waited = !(hp && hp->all_arrived);
    auto wait_input = [&]() -> cudaError_t {  // the caller's stream after the last input slice (host entry points)
        if (input_waited) return cudaSuccess;
        input_waited = true;
        return cudaStreamWaitEvent(st, hp->all_arrived, 0);
    };
    auto join_side = [&]() -> cudaError_t {
        if (!ctx->side_pending) return cudaSuccess;
        ctx->side_pending = false;
        return cudaStreamWaitEvent(st, ctx->ev_join, 0);
    };

    // ---- workspace plan ----
    const i64 R = ws.left() - 8192;
    // a window of the candidate buffer ends with a whole record's pairs: at most one per other sequence
    const i64 cslack = n_total + 64;
    i64 ccap = ctx->opt_cand_cap > 0 ? ctx->opt_cand_cap : std::max<i64>(1 << 20, std::min<i64>(2 * nmax, nmax / 2 + ((i64)128 << 20)));
    // Survivor list of multi-flush searches: never smaller than the caller's capacity (+ a little).  A pair found in
    // several chunks or windows is appended once per flush; when an append does not fit, the list is sorted,
    // deduplicated and cut to its smallest `capacity` entries, and the flush is repeated (see the window loop).
    const i64 scap_min = capacity + 4096;
    i64 scap = std::max<i64>(std::max<i64>(1 << 20, nmax / 4), scap_min + (ctx->opt_cand_cap > 0 ? ccap : 0));
    if (ctx->opt_surv_cap > 0) scap = std::max<i64>(scap_min, ctx->opt_surv_cap);
    i64 ncap = std::max<i64>(nmax, 1);
    u32 P = ctx->opt_force_chunks > 0 ? (u32)ctx->opt_force_chunks : 1;
    // A chunk carries fewer than 2^30 records (30-bit cursors and counts): a larger search is split up front, into chunks
    // expected to hold <= 3/4 * 2^30, so that the record buffers and the fused plan (bins, buckets) are sized for a chunk
    // and not for the whole (sized for the whole, the buckets would outgrow the join's stage and every chunk would take
    // the exact pipeline).
    if (ctx->opt_force_chunks <= 0 && nmax >= ((i64)3 << 28)) P = (u32)((nmax + ((i64)3 << 28) - 1) / ((i64)3 << 28));
    if (P > 1) ncap = std::min<i64>(nmax, nmax / P + nmax / (4 * P) + 4096);
    if (rec_bytes(ncap, npass_max) + cand_bytes(ccap + cslack, ppass) + cand_bytes(scap, spass) > R) {
        if (ctx->opt_cand_cap <= 0) ccap = std::min<i64>(ccap, std::max<i64>(4096, R / 4 / 17 - cslack));
        scap = std::min<i64>(scap, std::max<i64>(scap_min, R * 15 / 100 / 17));
        const i64 rrem = R - cand_bytes(ccap + cslack, ppass) - cand_bytes(scap, spass);
        if (rrem <= 0) return SYMDEL_E_WORKSPACE;
        // largest ncap that fits in rrem (16 B/record + ~0.26 B/record of tile status per pass)
        i64 lo = 0, hi = ncap;
        while (lo < hi) {
            i64 mid = (lo + hi + 1) / 2;
            if (rec_bytes(mid, npass_max) <= rrem) lo = mid; else hi = mid - 1;
        }
        ncap = lo;
        if (ncap < 4096) return SYMDEL_E_WORKSPACE;
        if (ctx->opt_force_chunks <= 0) P = (u32)std::max<i64>(1, (nmax + nmax / 8 + ncap - 1) / ncap);
    }
    const FusedPlan fp = plan_fused(ncap);
    u64* recA = ws.take<u64>(std::max(ncap, fp.bins_rec));
    u64* recB = ws.take<u64>(std::max(ncap, fp.bkt_rec));
    u32 *cur1 = fcnt, *cnt2 = fcnt + 256;
    void* rec_scratch = ws.take<char>(sd_sort_scratch_bytes(ncap, npass_max));
    u64* tile_prefix = ws.take<u64>(2 * sd_join_tiles(ncap) + 2);
    const i64 cphys = ccap + cslack;
    u64* candA = ws.take<u64>(cphys);
    u64* candB = ws.take<u64>(cphys);
    void* cand_scratch = ws.take<char>(sd_sort_scratch_bytes(cphys, ppass));
    u64* verify_lb = ws.take<u64>(cphys / 256 + 2);
    u64* survA = ws.take<u64>(scap);
    u64* survB = ws.take<u64>(scap);
    void* surv_scratch = ws.take<char>(sd_sort_scratch_bytes(scap, spass));
    u64* final_lb = ws.take<u64>(scap / 256 + 2);
    if (!ws.ok) return SYMDEL_E_WORKSPACE;

    const int width = (prefix > 0 ? std::min(maxlen, prefix) : maxlen) + 1;  // generation works on the (truncated) sequences
    i64 n_surv = 0, flushes = 0, surv_lower_bound = 0;
    // S5 as SURVEY.md section 8(a) words it: the chunks of the fused pipeline APPEND their candidates to one window, and the
    // window is deduplicated and verified "when the candidate buffer fills, or after the last chunk" — not once per chunk.
    // acc = candidates of earlier chunks waiting in candA[0, acc); acc_rec = the records they came from.
    bool accumulate = !ctx->opt_flush_per_chunk;
    i64 acc = 0, acc_rec = 0;
    bool direct = false;  // the single flush wrote the outputs itself
    enum { ST_GEN, ST_SORT, ST_EMIT, ST_DEDUP, ST_VERIFY };
    i64 pass_count = 0;

restart:
    if (P > 65536) return SYMDEL_E_WORKSPACE;
    tm.spans.clear();
    pass_count = 0;
    n_surv = 0;
    flushes = 0;
    surv_lower_bound = 0;
    direct = false;
    acc = acc_rec = 0;
    S.n_records = S.n_candidates = 0;
    lay.n_chunks = P;
    if (!info_fresh) CK(cudaMemsetAsync(&info->n_surv, 0, sizeof(u64) * 3, st));  // n_surv, n_out, n_unique
    for (u32 c = 0; c < P; ++c) {
        lay.chunk = c;
        lay.chunk_lo = chunk_pos(c, P);
        lay.chunk_hi = chunk_pos(c + 1, P);
        bool chunk_exact = false;  // a windowed fused search met a bucket whose pairs exceed a whole window: the chunk is redone by the exact pipeline
    redo_chunk:
        // ---- fused pipeline: generation + level-1 partition, level-2 partition, bucket join ----
        bool fused_ok = false, fused_more = false;  // fused_more: buckets whose pairs did not fit the window wait for the next pass
        i64 C = 0, wend = 0, N = 0;
        const u64* f_bkt = nullptr;
        u32* f_bcnt = nullptr;
        u32 f_bcap = 0, f_nb = 0;
        // (a chunk expected to hold 2^30 records or more goes to the exact pipeline, which splits it further)
        if (!chunk_exact && !ctx->opt_exact && ctx->opt_sort_bits < 0 && !ctx->opt_join_general && lay.hash_bits >= fp.b &&
            nmax / (i64)P < ((i64)1 << 30) && fp.cap2 <= sd_join_bkt_max_cap() && 64 - (lay.id_bits + lay.hash_bits) + fp.b >= sd_join_bkt_link_bits((u32)fp.cap2) &&
            sd_gen_part_applies(lay, width)) {
            const size_t x0 = tm.mark();
            lay.sort_bits = fp.b;
            if (!info_fresh) CK(cudaMemsetAsync(&info->part_overflow, 0, sizeof(u32), st));
            const int fresh = info_fresh ? 1 : 0;
            info_fresh = false;
            // level-1 cursors and level-2 counts are neighbours: one clear for both, ahead of generation
            CK(cudaMemsetAsync(fcnt, 0, (size_t)(256 + (fp.b2 ? fp.nbuckets : 0)) * sizeof(u32), st));
            const double rpr = (double)nmax / (double)std::max<i64>(residues, 1) / (double)P, avg_len = (double)residues / (double)n_total;
            // Query filter (cross-search with the queries the small side): set A is generated first, its records mark a bitmap per
            // level-1 bin, and the level-2 partition drops the set-B records that no set-A record can match (radix_sort.cu).
            // The bitmaps live in the second candidate buffer, which nothing uses before the candidate sort.
            int fbits = 0;
            u32 *fbm = nullptr, *cnt_a = nullptr;
            const int fshift_top = lay.id_bits + lay.hash_bits - 8;
            if (cross && fp.b2 && !ctx->opt_no_query_filter && A.n * 4 <= B.n && sd_gen_part_sliceable(lay, width)) {
                const double a_per_bin = (double)(nmax - (i64)ctx->h_info->nmax_b) / (double)P / 256.0;
                fbits = 13;
                while (fbits < SD_FBITS_MAX && (double)((i64)1 << fbits) < 6.0 * a_per_bin) ++fbits;
                const i64 need = ((i64)256 << (fbits - 5)) * 4 + 256 * 4;
                if (2.0 * a_per_bin > (double)((i64)1 << fbits) || lay.hash_bits < 8 + fbits || need > cphys * 8) fbits = 0;  // (too dense to pay, or no room)
                if (fbits) fbm = reinterpret_cast<u32*>(candB), cnt_a = fbm + ((size_t)256 << (fbits - 5));
            }
            S.query_filter_bits = fbits;
            if (fbits) {
                CK(wait_input());
                CK(sd_gen_part(A, B, lay, width, recA, cur1, (u64)fp.cap1, rpr, avg_len, 0, -2, 1, info, st, &S.n_launches));
                CK(cudaMemcpyAsync(cnt_a, cur1, 256 * sizeof(u32), cudaMemcpyDeviceToDevice, st));
                CK(sd_bin_bitmap(recA, cnt_a, fp.cap1, fbm, fbits, fshift_top - fbits, st, &S.n_launches));
                CK(sd_gen_part(A, B, lay, width, recA, cur1, (u64)fp.cap1, rpr, avg_len, 0, -3, 1, info, st, &S.n_launches));
            } else
            if (hp && hp->n_slices > 1 && !input_waited && sd_gen_part_sliceable(lay, width)) {
                // generation follows the input slice by slice: slice i is generated while slice i + 1 is being copied
                i64 t0 = 0;
                for (int i = 0; i < hp->n_slices; ++i) {
                    CK(cudaStreamWaitEvent(st, hp->arrived[i], 0));
                    CK(sd_gen_part(A, B, lay, width, recA, cur1, (u64)fp.cap1, rpr, avg_len, t0, hp->task_end[i], 1, info, st, &S.n_launches));
                    t0 = hp->task_end[i];
                }
                input_waited = true;
            } else {
                CK(wait_input());
                CK(sd_gen_part(A, B, lay, width, recA, cur1, (u64)fp.cap1, rpr, avg_len, 0, -1, 1, info, st, &S.n_launches));
            }
            const size_t x1 = tm.mark();
            if (fp.b2)
                CK(sd_part2(recA, cur1, fp.cap1, recB, cnt2, fp.cap2, fp.b2, lay.id_bits + lay.hash_bits - fp.b, 1, fbm, cnt_a, fbits, fshift_top - fbits, info, st,
                            &S.n_launches));
            const size_t x2 = tm.mark();
            f_bkt = fp.b2 ? recB : recA;
            f_bcnt = fp.b2 ? cnt2 : cur1;
            f_bcap = (u32)(fp.b2 ? fp.cap2 : fp.cap1), f_nb = (u32)fp.nbuckets;
            u32* h_cur = reinterpret_cast<u32*>(ctx->h_info + 1);
            CK(sd_join_bkt(f_bkt, f_bcnt, f_bcap, f_nb, lay, candA, (u64)ccap, 1, fresh, fbits ? 1 : 0, acc > 0 ? 1 : 0, info, st, &S.n_launches));
            CK(join_side());
            CK(cudaMemcpyAsync(h_cur, cur1, 256 * sizeof(u32), cudaMemcpyDeviceToHost, st));  // (bit 31 of a count is the join's "open" mark)
            rc = read_info(ctx, info, st);
            if (rc) return rc;
            if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
            // pairs beyond one window: the buckets that fit are done, the others are joined by later passes (window loop below)
            fused_more = ctx->h_info->join_fallback != 0;
            C = (i64)std::min<u64>(ctx->h_info->n_cand, ~ctx->h_info->nofit_inv);
            // (nothing written and buckets left open: one bucket's pairs exceed a whole window — unless the small join instance was
            //  preferred and simply could not stage any bucket: then the next pass, with the large instance, decides)
            fused_ok = !ctx->h_info->part_overflow && !(fused_more && C == 0 && !fbits);
            if (!fused_ok && acc > 0) {  // (a full bin with candidates of earlier chunks still pending: start over, one flush per chunk)
                accumulate = false;
                goto restart;
            }
            if (!fused_ok) fused_more = false, C = 0;
            if (fused_ok) {
                for (int i = 0; i < 256; ++i) N += h_cur[i] & 0x7fffffffu;
                wend = C;
                const size_t x3 = tm.mark();
                tm.span(ST_GEN, x0, x1);
                tm.span(ST_SORT, x1, x2);
                tm.span(ST_EMIT, x2, x3);
                pass_count += fp.b2 ? 1 : 0;
                S.sort_pass_records = N;
                S.sort_bits = fp.b;
                S.n_records += N;
                S.n_candidates += C - acc;  // (C counts the pending candidates of earlier chunks too)
                ++S.fused_chunks;
                // every pair of this chunk is in the window and there is room for about as many again: the flush waits
                if (accumulate && !fused_more && c + 1 < P && C + 2 * (C - acc) <= ccap) {
                    acc = C;
                    acc_rec += N;
                    continue;
                }
            }
        }
        u64* sorted = nullptr;
        if (!fused_ok) {
        const size_t e0 = tm.mark();
        info_fresh = false;
        CK(wait_input());
        // ---- S1: count, scan, generate ----
        CK(sd_count(A, B, lay, width, cnt, info, st, &S.n_launches));
        CK(sd_scan_counts(cnt, n_total, rec_off, scan_lb, info, st, &S.n_launches));
        CK(join_side());
        rc = read_info(ctx, info, st);
        if (rc) return rc;
        if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);  // (k_pack's residue check is in by now: no generation, no re-chunking on bad input)
        N = (i64)ctx->h_info->n_records;
        if (N > ncap || N >= ((i64)1 << 30)) {
            if (ctx->opt_force_chunks > 0 && N <= ncap) return SYMDEL_E_TOO_MANY;
            P *= 2;
            goto restart;
        }
        S.n_records += N;
        if (N == 0) continue;
        lay.sort_bits = pick_sort_bits(N);
        S.sort_bits = lay.sort_bits;
        const int npass = lay.sort_bits / 8;
        const int sort_begin = lay.id_bits + lay.hash_bits - lay.sort_bits;  // first radix-partitioned bit of a record
        CK(sd_sort_prepare(rec_scratch, N, npass, st));
        CK(sd_generate(A, B, lay, width, rec_off, recA, sd_sort_hist_ptr(rec_scratch), sort_begin, npass, info, st,
                       &S.n_launches));
        CK(sd_sort_hist_scan(rec_scratch, npass, st, &S.n_launches));
        const size_t e1 = tm.mark();
        // ---- S2: radix partition on the top sort_bits (exactly npass onesweep launches between e1 and e2) ----
        CK(sd_sort_passes(recA, recB, N, nullptr, sort_begin, npass, ctx->opt_sort_stable ? 1 : 0, (int)ctx->opt_sort_variant, rec_scratch, st, &sorted,
                          &S.n_launches));
        const size_t e2 = tm.mark();
        // ---- S3a: join (first window): the fast kernel when everything fits one window, else the general one ----
        bool general = ctx->opt_join_general != 0;
        if (!general) {
            CK(sd_join_fast(sorted, N, lay, candA, (u64)ccap, (u32*)tile_prefix, info, st, &S.n_launches));
            rc = read_info(ctx, info, st);
            if (rc) return rc;
            if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
            if (ctx->h_info->join_redo && !ctx->h_info->join_fallback) {  // dense tiles: the large-list instance
                S.join_redo_tiles += ctx->h_info->join_redo;
                CK(sd_join_fast_redo(sorted, N, lay, candA, (u64)ccap, (const u32*)tile_prefix, ctx->h_info->join_redo, info, st,
                                     &S.n_launches));
                rc = read_info(ctx, info, st);
                if (rc) return rc;
            }
            general = ctx->h_info->join_fallback != 0;
            ctx->h_info->win_end = ctx->h_info->n_cand;
        }
        if (general) {
            ++S.join_general;
            CK(sd_join(sorted, N, lay, candA, (u64)cphys, 0, (u64)ccap, 1, tile_prefix, info, st, &S.n_launches));
            rc = read_info(ctx, info, st);
            if (rc) return rc;
            if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
        }
        C = (i64)ctx->h_info->n_cand;
        wend = (i64)ctx->h_info->win_end;
        S.n_candidates += C;
        const size_t e3 = tm.mark();
        tm.span(ST_GEN, e0, e1);
        tm.span(ST_SORT, e1, e2);
        tm.span(ST_EMIT, e2, e3);
        pass_count += npass;
        S.sort_pass_records = N;
        }  // exact pipeline
        for (i64 w0 = 0; w0 < C || fused_more;) {
            const size_t f0 = tm.mark();
            if (fused_ok && (w0 > 0 || C == 0)) {
                // ---- next pass of the bucket join: the buckets not marked done, into a fresh window ----
                CK(sd_join_bkt(f_bkt, f_bcnt, f_bcap, f_nb, lay, candA, (u64)ccap, 0, 0, 0, 0, info, st, &S.n_launches));
                rc = read_info(ctx, info, st);
                if (rc) return rc;
                if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
                fused_more = ctx->h_info->join_fallback != 0;
                const i64 X = (i64)std::min<u64>(ctx->h_info->n_cand, ~ctx->h_info->nofit_inv);
                if (fused_more && X == 0) {  // one bucket's pairs exceed a whole window (what was appended so far stays: the final pass removes repeats)
                    chunk_exact = true;
                    S.n_records -= N;
                    --S.fused_chunks;
                    ++flushes;  // (forces the final sort + unique even if nothing else is flushed twice)
                    goto redo_chunk;
                }
                C += X;
                wend = w0 + X;
                S.n_candidates += X;
                ++S.join_windows;
                if (X == 0) break;  // the remaining buckets had no pairs
            } else if (w0 > 0) {
                CK(sd_join(sorted, N, lay, candA, (u64)cphys, (u64)w0, (u64)(w0 + ccap), 0, tile_prefix, info, st,
                           &S.n_launches));
                rc = read_info(ctx, info, st);
                if (rc) return rc;
                if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
                wend = (i64)ctx->h_info->win_end;
            }
            const i64 nc = wend - w0;  // the records that start in [w0, w0 + ccap), whole
            if (nc <= 0 || nc > cphys) return SYMDEL_E_INTERNAL;
            const size_t f1 = tm.mark();
            // ---- S3b: sort the packed pair ids ----
            CK(sd_sort_prepare(cand_scratch, nc, ppass, st));
            u64* csorted = nullptr;
            const u64* nc_dev = nullptr;  // where the number of candidates to sort and verify lives (nullptr: nc)
            // The filter pays when the sort is throughput-bound and the distinct pairs (the table lines it touches) stay
            // cache-resident: config 5 (16.8 M candidates, 0.9 M distinct) 0.77 -> 0.42 ms; config 3 (3.7 M) 0.24 -> 0.21 ms;
            // dense 1 M (74 M candidates, 24 M distinct): the table misses L2, 3.8 -> 5.0 ms.
            const bool use_filter = ctx->opt_cand_filter == 1 || (ctx->opt_cand_filter == 0 && nc >= ((i64)1 << 20) && nc < (N + acc_rec) / 4);
            if (use_filter) {
                // duplicate suppression before the sort: a best-effort hash set in a record buffer that is free now
                // (fused: the level-1 bins; exact: the ping-pong buffer that does not hold the partitioned records)
                const bool in_b = fused_ok ? fp.b2 == 0 : sorted == recA;  // fused: the buckets (recB, or recA without a level 2) may be joined again
                u64* table = in_b ? recB : recA;
                const i64 table_room = in_b ? std::max(ncap, fp.bkt_rec) : std::max(ncap, fp.bins_rec);
                int tb = 16;
                while (tb < 27 && ((i64)1 << tb) < nc) ++tb;
                while (tb > 10 && ((i64)1 << tb) > table_room) --tb;
                CK(cudaMemsetAsync(table, 0, (size_t)8 << tb, st));
                CK(sd_cand_filter(candA, nc, table, tb, candB, &info->n_filt, ppass, cand_scratch, st, &S.n_launches));
                CK(sd_sort_hist_scan(cand_scratch, ppass, st, &S.n_launches));
                nc_dev = &info->n_filt;
                CK(sd_sort_passes(candB, candA, nc, nc_dev, 0, ppass, 0, (int)ctx->opt_sort_variant, cand_scratch, st, &csorted,
                                  &S.n_launches));
            } else {
                CK(sd_sort_histogram(candA, nc, 0, ppass, cand_scratch, st, &S.n_launches));
                CK(sd_sort_hist_scan(cand_scratch, ppass, st, &S.n_launches));
                CK(sd_sort_passes(candA, candB, nc, nullptr, 0, ppass, 0, (int)ctx->opt_sort_variant, cand_scratch, st, &csorted,
                                  &S.n_launches));
            }
            const size_t f2 = tm.mark();
            // ---- S4: unique + verify; survivors appended at n_surv — or, when this window holds every candidate of
            //      the only chunk, unpacked straight into the outputs (no survivor list, no finalize) ----
            direct = c + 1 == P && w0 == 0 && wend == C && !fused_more && flushes == 0;  // (earlier chunks, if any, are all in this window)
            if (direct)
                CK(sd_verify_direct(csorted, nc, nc_dev, slots, lay, maxlen, out_i, out_j, out_dist, capacity, verify_lb, info, st,
                                    &S.n_launches));
            else {
                // sort the survivor list, drop the repeats, keep the smallest `capacity`: makes room for the next append
                auto merge_survivors = [&]() -> int {
                    CK(sd_sort_prepare(surv_scratch, n_surv, spass, st));
                    CK(sd_sort_histogram(survA, n_surv, 3, spass, surv_scratch, st, &S.n_launches));
                    CK(sd_sort_hist_scan(surv_scratch, spass, st, &S.n_launches));
                    u64* ssorted = nullptr;
                    CK(sd_sort_passes(survA, survB, n_surv, nullptr, 3, spass, 0, (int)ctx->opt_sort_variant, surv_scratch, st, &ssorted,
                                      &S.n_launches));
                    u64* dst = ssorted == survA ? survB : survA;
                    CK(sd_finalize(ssorted, n_surv, lay, 1, nullptr, nullptr, nullptr, dst, scap, final_lb, info, st, &S.n_launches));
                    int r = read_info(ctx, info, st);
                    if (r) return r;
                    const i64 uniq = (i64)ctx->h_info->n_out;
                    if (uniq > capacity) surv_lower_bound = std::max(surv_lower_bound, uniq);  // the result exceeds `capacity`
                    n_surv = std::min(uniq, capacity);
                    if (dst != survA) std::swap(survA, survB);
                    ++S.surv_merges;
                    return SYMDEL_OK;
                };
                bool merged = false;
                if (n_surv > scap / 2 && n_surv + nc > scap) {  // likely not to fit: merge first
                    if ((rc = merge_survivors())) return rc;
                    merged = true;
                }
                // v0 / vn: the slice [v0, v0 + vn) of the sorted window that the next sd_verify takes (the whole window
                // unless an overflow forces slices); vtotal: candidates in the window once it is known on the host
                i64 v0 = 0, vn = nc, vtotal = nc;
                const u64* vdev = nc_dev;
                bool sliced = false;
                for (;;) {
                    CK(cudaMemsetAsync(&info->surv_overflow, 0, sizeof(u32), st));
                    CK(sd_verify(csorted + v0, vn, vdev, slots, lay, maxlen, survA, (u64)n_surv, (u64)scap, verify_lb, info, st,
                                 &S.n_launches));
                    rc = read_info(ctx, info, st);
                    if (rc) return rc;
                    if (!ctx->h_info->surv_overflow) {
                        v0 += vn;
                        if (!sliced || v0 >= vtotal) break;
                        // next slice: cut the list back to <= `capacity` entries first, so that the slice fits whatever it yields
                        n_surv = (i64)ctx->h_info->n_surv;
                        if (n_surv > 0 && (rc = merge_survivors())) return rc;
                        vn = std::min<i64>(vtotal - v0, scap - n_surv);
                        continue;
                    }
                    // the survivors did not fit behind the list (nothing was lost, n_surv stands): merge the list once ...
                    if (!merged && n_surv > 0) {
                        if ((rc = merge_survivors())) return rc;
                        merged = true;
                        continue;
                    }
                    // ... and if the list is as short as it gets (<= `capacity` entries of scap >= capacity + 4096) and the window
                    // still yields more than the room behind it, verify the window in slices of at most that room: a candidate
                    // gives at most one survivor, so a slice always fits.  The merges between slices keep the smallest `capacity`
                    // pairs and the count of distinct pairs seen (surv_lower_bound), which is what SYMDEL_E_CAPACITY reports.
                    if (vdev) vtotal = (i64)ctx->h_info->n_filt, vdev = nullptr;
                    if (scap - n_surv <= 0) return SYMDEL_E_INTERNAL;
                    vn = std::min<i64>(vtotal - v0, scap - n_surv);
                    sliced = true;
                }
                if (sliced) ++flushes;  // (a repeated pair may straddle two slices: the final pass has to sort and deduplicate)
            }
            rc = read_info(ctx, info, st);
            if (rc) return rc;
            if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
            n_surv = (i64)ctx->h_info->n_surv;
            const size_t f3 = tm.mark();
            tm.span(ST_EMIT, f0, f1);
            tm.span(ST_DEDUP, f1, f2);
            tm.span(ST_VERIFY, f2, f3);
            ++flushes;
            acc = acc_rec = 0;
            w0 = wend;
        }
    }
    if (acc > 0) return SYMDEL_E_INTERNAL;  // (the last chunk always flushes)

    // ---- final: (sort + unique) and unpack ----
    const size_t g0 = tm.mark();
    i64 n_out = 0;
    if (direct) {
        n_out = (i64)ctx->h_info->n_out;
    } else if (n_surv > 0) {
        const u64* fin = survA;
        if (flushes > 1) {
            CK(sd_sort_prepare(surv_scratch, n_surv, spass, st));
            CK(sd_sort_histogram(survA, n_surv, 3, spass, surv_scratch, st, &S.n_launches));
            CK(sd_sort_hist_scan(surv_scratch, spass, st, &S.n_launches));
            u64* ssorted = nullptr;
            CK(sd_sort_passes(survA, survB, n_surv, nullptr, 3, spass, 0, (int)ctx->opt_sort_variant, surv_scratch, st, &ssorted, &S.n_launches));
            fin = ssorted;
        }
        CK(sd_finalize(fin, n_surv, lay, flushes > 1 ? 1 : 0, out_i, out_j, out_dist, nullptr, capacity, final_lb, info, st,
                       &S.n_launches));
        rc = read_info(ctx, info, st);
        if (rc) return rc;
        // (after a merge that cut the list to `capacity` entries the exact count is not known any more: the
        //  number of distinct pairs seen at that point is a lower bound, and it exceeds `capacity`)
        n_out = std::max<i64>((i64)ctx->h_info->n_out, surv_lower_bound);
    }
    const size_t g1 = tm.mark();
    if (tm.on) {
        CK(cudaStreamSynchronize(st));
        S.ms_prepare = tm.ms(ev_begin, ev_prepared);
        S.ms_generate = tm.total(ST_GEN);
        S.ms_sort = tm.total(ST_SORT);
        S.ms_emit = tm.total(ST_EMIT);
        S.ms_dedup = tm.total(ST_DEDUP);
        S.ms_verify = tm.total(ST_VERIFY) + tm.ms(g0, g1);
        S.ms_total = tm.ms(ev_begin, g1);
        S.ms_sort_pass_avg = pass_count ? S.ms_sort / (float)pass_count : 0.f;
    }
    S.n_unique = (i64)ctx->h_info->n_unique;
    S.n_outputs = n_out;
    S.n_chunks = P;
    S.n_flushes = flushes;
    *n_pairs_host = n_out;
    return n_out > capacity ? SYMDEL_E_CAPACITY : SYMDEL_OK;
}

// Every way out of the pipeline leaves the caller's stream ordered after the side stream's work (which reads and
// writes the caller's workspace): a caller may release the workspace in stream order right after the call.
int run_pipeline(symdel_ctx* ctx, SeqSetDev A, SeqSetDev B, int cross, int d, void* workspace, i64 workspace_bytes, i32* out_i,
                 i32* out_j, i32* out_dist, i64 capacity, i64* n_pairs_host, cudaStream_t st, const HostPlan* hp = nullptr) {
    const int rc = run_pipeline_body(ctx, A, B, cross, d, workspace, workspace_bytes, out_i, out_j, out_dist, capacity, n_pairs_host, st, hp);
    if (ctx && ctx->side_pending) {
        ctx->side_pending = false;
        if (cudaStreamWaitEvent(st, ctx->ev_join, 0) != cudaSuccess) cudaStreamSynchronize(ctx->side);
    }
    return rc;
}

int ensure_arena(symdel_ctx* ctx, void** arena, size_t* have, size_t bytes) {
    if (*have >= bytes) return SYMDEL_OK;
    if (*arena) cudaFree(*arena);
    *arena = nullptr;
    *have = 0;
    CK(cudaMalloc(arena, bytes));
    *have = bytes;
    return SYMDEL_OK;
}

int run_host(symdel_ctx* ctx, const int8_t* a_seqs, const i64* a_off, i64 n_a, const int8_t* b_seqs, const i64* b_off,
             i64 n_b, int cross, int d, i32* out_i, i32* out_j, i32* out_dist, i64 capacity, i64* n_pairs_host) {
    if (!ctx || !n_pairs_host || n_a < 0 || n_b < 0 || d < 0 || d > SD_D_MAX || capacity < 0) return SYMDEL_E_ARG;
    *n_pairs_host = 0;
    if (n_a == 0 || (cross && n_b == 0)) {
        ctx->stats = symdel_stats{};
        return SYMDEL_OK;
    }
    if (!a_seqs || !a_off || (cross && (!b_seqs || !b_off))) return SYMDEL_E_ARG;
    if (a_off[0] != 0 || (cross && b_off[0] != 0)) return SYMDEL_E_OFFSETS;
    CK(cudaSetDevice(ctx->device));
    const i64 res_a = a_off[n_a], res_b = cross ? b_off[n_b] : 0;
    if (res_a < 0 || res_b < 0) return SYMDEL_E_OFFSETS;
    // ---- inputs first: the copies run (on the side stream) while the host does S0 on its own copy of the offsets and sizes
    //      the workspace; a large self-search is sent in slices so that generation can start when the first has arrived ----
    const i64 in_bytes = align_up(res_a + 16) + align_up((n_a + 1) * 8) + align_up(res_b + 16) + align_up((n_b + 1) * 8);
    int rc = ensure_arena(ctx, &ctx->in_arena, &ctx->in_arena_bytes, (size_t)(in_bytes + 4096));
    if (rc) return rc;
    cudaStream_t st = ctx->stream, cs = ctx->side;
    Bump in(ctx->in_arena, (i64)ctx->in_arena_bytes);
    int8_t* d_as = in.take<int8_t>(res_a + 16);
    i64* d_ao = in.take<i64>(n_a + 1);
    int8_t* d_bs = in.take<int8_t>(res_b + 16);
    i64* d_bo = in.take<i64>(n_b + 1);
    if (!in.ok) return SYMDEL_E_INTERNAL;
    while (ctx->hp_events.size() < (size_t)HP_MAX_SLICES + 2) {
        cudaEvent_t e;
        CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->hp_events.push_back(e);
    }
    HostPlan hp;
    // (the offsets are validated on the device, by k_prepare; here they only place the slice boundaries, clamped: the
    //  copies never leave the context's own arena)
    auto clampi = [](i64 x, i64 lo, i64 hi) { return x < lo ? lo : (x > hi ? hi : x); };
    CK(cudaMemcpyAsync(d_ao, a_off, (size_t)(n_a + 1) * 8, cudaMemcpyHostToDevice, cs));
    if (cross) CK(cudaMemcpyAsync(d_bo, b_off, (size_t)(n_b + 1) * 8, cudaMemcpyHostToDevice, cs));
    hp.offsets_arrived = ctx->hp_events[HP_MAX_SLICES + 1];
    CK(cudaEventRecord(hp.offsets_arrived, cs));
    const i64 tasks_a = (n_a + 31) / 32;
    hp.n_slices = (!cross && n_a >= 65536) ? 4 : 1;  // (config 3 end to end: 2 slices 2.04 ms, 4: 2.02, 6: 2.09, 8: 2.11)
    {
        i64 s0 = 0;
        for (int i = 0; i < hp.n_slices; ++i) {
            hp.task_end[i] = tasks_a * (i + 1) / hp.n_slices;
            const i64 s1 = std::min<i64>(n_a, hp.task_end[i] * 32);
            const i64 r0 = clampi(a_off[s0], 0, res_a), r1 = clampi(a_off[s1], r0, res_a);
            if (r1 > r0) CK(cudaMemcpyAsync(d_as + r0, a_seqs + r0, (size_t)(r1 - r0), cudaMemcpyHostToDevice, cs));
            hp.arrived[i] = ctx->hp_events[i];
            CK(cudaEventRecord(hp.arrived[i], cs));
            s0 = s1;
        }
    }
    if (cross && res_b) CK(cudaMemcpyAsync(d_bs, b_seqs, (size_t)res_b, cudaMemcpyHostToDevice, cs));
    hp.all_arrived = ctx->hp_events[HP_MAX_SLICES];
    CK(cudaEventRecord(hp.all_arrived, cs));
    // Workspace: sized from an ESTIMATE of the record count (every sequence as long as the mean, rounded up, plus one) — no
    // pass over a million host offsets on the critical path.  If the estimate is low the planner cuts the search into key-range
    // chunks: slower, never wrong.  The exact count is S0's, on the device.
    const i64 pfx = ctx->opt_prefix > 0 ? ctx->opt_prefix : SD_L_MAX;
    auto est = [&](i64 n, i64 res) -> i64 {
        if (n <= 0) return 0;
        const i64 Lm = std::min<i64>(std::min<i64>((res + n - 1) / n + 1, pfx), SD_L_MAX);
        return n * (i64)vcount_host((int)Lm, d);
    };
    i64 nmax = est(n_a, res_a) + est(n_b, res_b);
    const i64 n_total = n_a + n_b;
    const int npass_max = 7, ppass_max = 8;
    const i64 out_bytes = 3 * align_up(capacity * 4 + 16);
    i32 *d_i = nullptr, *d_j = nullptr, *d_d = nullptr;
    for (int attempt = 0;; ++attempt) {
        const i64 ccap = std::max<i64>(1 << 20, std::min<i64>(2 * nmax, nmax / 2 + ((i64)128 << 20))), scap = std::max<i64>(std::max<i64>(1 << 20, nmax / 4), capacity);
        const i64 ws_bytes = fixed_bytes(n_total) + rec_bytes(std::max<i64>(nmax, 1), npass_max) + cand_bytes(ccap + n_total + 64, ppass_max) +
                             cand_bytes(scap, ppass_max) + 65536;
        rc = ensure_arena(ctx, &ctx->arena, &ctx->arena_bytes, (size_t)(out_bytes + ws_bytes + 4096));
        if (rc) break;
        Bump ar(ctx->arena, (i64)ctx->arena_bytes);
        d_i = ar.take<i32>(capacity + 4);
        d_j = ar.take<i32>(capacity + 4);
        d_d = ar.take<i32>(capacity + 4);
        // (an arena left larger by an earlier call is used whole: more room never hurts the plan)
        const i64 ws_have = std::max<i64>(ws_bytes, (ar.left() - 4096) / 256 * 256);
        void* d_ws = ar.take<char>(ws_have);
        if (!ar.ok) {
            rc = SYMDEL_E_INTERNAL;
            break;
        }
        SeqSetDev A{d_as, d_ao, n_a}, B{d_bs, d_bo, cross ? n_b : 0};
        rc = run_pipeline(ctx, A, B, cross, d, d_ws, ws_have, d_i, d_j, d_d, capacity, n_pairs_host, st, &hp);
        if (rc != SYMDEL_E_WORKSPACE || attempt > 0) break;
        // The estimate was too low even for a chunked search (lengths far from their mean, or an output capacity that
        // leaves no room): size the arena from the exact count — one pass over the host offsets, this once — and repeat.
        i64 exact = 0;
        bool bad = false;
        for (int sset = 0; sset < (cross ? 2 : 1); ++sset) {
            const i64* off = sset ? b_off : a_off;
            const i64 n = sset ? n_b : n_a;
            u64 vtab[SD_L_MAX + 1];
            for (int L = 0; L <= SD_L_MAX; ++L) vtab[L] = vcount_host((int)std::min<i64>(L, pfx), d);
            for (i64 i = 0; i < n; ++i) {
                const i64 L = off[i + 1] - off[i];
                if (L < 0 || L > SD_L_MAX) bad = true;
                else exact += (i64)vtab[L];
            }
        }
        if (bad || exact <= nmax) break;  // (malformed offsets are reported by the device pass; nothing to gain otherwise)
        nmax = exact;
    }
    if (rc != SYMDEL_OK && rc != SYMDEL_E_CAPACITY) {
        cudaStreamSynchronize(cs);  // (an early way out may not have waited for the copies: the caller's buffers are free on return)
        return rc;
    }
    const i64 ncopy = std::min<i64>(*n_pairs_host, capacity);
    if (ncopy > 0) {
        CK(cudaMemcpyAsync(out_i, d_i, (size_t)ncopy * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(out_j, d_j, (size_t)ncopy * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(out_dist, d_d, (size_t)ncopy * 4, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaStreamSynchronize(st));
    return rc;
}

}  // namespace

// =================================================================================================
extern "C" {

int symdel_create(symdel_ctx** out, int device) {
    if (!out) return SYMDEL_E_ARG;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return SYMDEL_E_CUDA;
    // The library is built for sm_100a only and its launch helpers size grids, warp tasks and shared-memory carve-outs for
    // the B200 (148 SMs, 227 KB of shared memory per block): any other device is refused here rather than mis-tuned.
    int cc_major = 0, cc_minor = 0, sms = 0, smem_optin = 0;
    if (cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&cc_minor, cudaDevAttrComputeCapabilityMinor, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) != cudaSuccess)
        return SYMDEL_E_CUDA;
    if (cc_major != 10 || cc_minor != 0 || sms != 148 || smem_optin < 232448) return SYMDEL_E_CUDA;
    symdel_ctx* ctx = new symdel_ctx();
    ctx->device = device;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->h_info, sizeof(DevInfo) + 256 * sizeof(u32));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) {
        // Constant tables and function attributes are per DEVICE: every context sets them up for its own device
        // (idempotent; serialised so that two threads creating contexts never interleave the uploads).
        static std::mutex setup_lock;
        std::lock_guard<std::mutex> g(setup_lock);
        e = sd_generate_setup();
        if (e == cudaSuccess) e = sd_sort_setup();
        if (e == cudaSuccess) e = sd_join_setup();
    }
    if (e != cudaSuccess) {
        symdel_destroy(ctx);
        return SYMDEL_E_CUDA;
    }
    *out = ctx;
    return SYMDEL_OK;
}

void symdel_destroy(symdel_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    if (ctx->arena) cudaFree(ctx->arena);
    if (ctx->in_arena) cudaFree(ctx->in_arena);
    if (ctx->h_info) cudaFreeHost(ctx->h_info);
    if (ctx->stream) cudaStreamDestroy(ctx->stream);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    for (auto e : ctx->events) cudaEventDestroy(e);
    for (auto e : ctx->hp_events) cudaEventDestroy(e);
    delete ctx;
}

int symdel_set_option(symdel_ctx* ctx, int option, int64_t value) {
    if (!ctx || value < 0) return SYMDEL_E_ARG;
    switch (option) {
        case SYMDEL_OPT_TIMING: ctx->opt_timing = value != 0; break;
        case SYMDEL_OPT_FORCE_CHUNKS: ctx->opt_force_chunks = value; break;
        case SYMDEL_OPT_CAND_CAPACITY: ctx->opt_cand_cap = value; break;
        case SYMDEL_OPT_HASH_BITS:
            if (value > 63) return SYMDEL_E_ARG;
            ctx->opt_hash_bits = value;
            break;
        case SYMDEL_OPT_SORT_BITS:
            if (value != 255 && (value % 8 != 0 || value > 56)) return SYMDEL_E_ARG;
            ctx->opt_sort_bits = value == 0 ? -1 : value == 255 ? 0 : value;
            break;
        case SYMDEL_OPT_SORT_STABLE: ctx->opt_sort_stable = value != 0; break;
        case SYMDEL_OPT_SORT_GROUPING: ctx->opt_sort_grouping = value != 0; break;
        case SYMDEL_OPT_JOIN_GENERAL: ctx->opt_join_general = value != 0; break;
        case SYMDEL_OPT_EXACT_PIPELINE: ctx->opt_exact = value != 0; break;
        case SYMDEL_OPT_METRIC:
            if (value > 1) return SYMDEL_E_ARG;
            ctx->opt_metric = value;
            break;
        case SYMDEL_OPT_PREFIX_LEN:
            if (value > SD_L_MAX) return SYMDEL_E_ARG;
            ctx->opt_prefix = value;
            break;
        case SYMDEL_OPT_NO_THINNING: ctx->opt_no_thinning = value != 0; break;
        case SYMDEL_OPT_GENERAL_GENERATE: ctx->opt_general_gen = value != 0; break;
        case SYMDEL_OPT_SURV_CAPACITY: ctx->opt_surv_cap = value; break;
        case SYMDEL_OPT_CAND_FILTER:
            if (value > 2) return SYMDEL_E_ARG;
            ctx->opt_cand_filter = value;
            break;
        case SYMDEL_OPT_NO_QUERY_FILTER: ctx->opt_no_query_filter = value != 0; break;
        case SYMDEL_OPT_FLUSH_PER_CHUNK: ctx->opt_flush_per_chunk = value != 0; break;
        case SYMDEL_OPT_SORT_VARIANT:
            if (value >= sd_sort_variants()) return SYMDEL_E_ARG;
            ctx->opt_sort_variant = value;
            break;
        default: return SYMDEL_E_ARG;
    }
    return SYMDEL_OK;
}

int symdel_get_stats(const symdel_ctx* ctx, symdel_stats* stats_host) {
    if (!ctx || !stats_host) return SYMDEL_E_ARG;
    *stats_host = ctx->stats;
    return SYMDEL_OK;
}

int symdel_last_cuda_error(const symdel_ctx* ctx) { return ctx ? (int)ctx->last_cuda : 0; }

const char* symdel_strerror(int code) {
    switch (code) {
        case SYMDEL_OK: return "ok";
        case SYMDEL_E_ARG: return "invalid argument";
        case SYMDEL_E_OFFSETS: return "offsets[0] != 0 or offsets not non-decreasing";
        case SYMDEL_E_TOO_LONG: return "a sequence is longer than SYMDEL_L_MAX";
        case SYMDEL_E_RESIDUE: return "residue code outside 1..31";
        case SYMDEL_E_TOO_MANY: return "too many sequences or records";
        case SYMDEL_E_WORKSPACE: return "workspace too small";
        case SYMDEL_E_CAPACITY: return "more result pairs than the output capacity";
        case SYMDEL_E_CUDA: return "CUDA error";
        case SYMDEL_E_INTERNAL: return "internal consistency check failed";
        case SYMDEL_E_STATIC_LIMIT: return "more keys than the built-in scratch of symdel_sort_u64_static holds (SYMDEL_STATIC_SORT_MAX_KEYS)";
        default: return "unknown error";
    }
}

int symdel_workspace_bytes(int64_t n_a, int64_t residues_a, int64_t n_b, int64_t residues_b, int max_len, int d,
                           int64_t capacity, int64_t* bytes_host) {
    if (!bytes_host || n_a < 0 || n_b < 0 || residues_a < 0 || residues_b < 0 || d < 0 || d > SD_D_MAX || max_len < 0 ||
        max_len > SD_L_MAX || capacity < 0)
        return SYMDEL_E_ARG;
    // V(L, d) <= 1 + L * (V(max_len, d) - 1) / max_len for L <= max_len
    const i64 n_total = n_a + n_b;
    const u64 vm = vcount_host(max_len, d);
    const i64 nbound = n_total + (max_len ? (i64)(((u64)(residues_a + residues_b) * (vm - 1) + max_len - 1) / max_len) : 0);
    const i64 ccap = std::max<i64>(1 << 20, std::min<i64>(2 * nbound, nbound / 2 + ((i64)128 << 20))), scap = std::max<i64>(std::max<i64>(1 << 20, nbound / 4), capacity);
    *bytes_host = fixed_bytes(n_total) + rec_bytes(std::max<i64>(nbound, 1), 7) + cand_bytes(ccap + n_total + 64, 8) + cand_bytes(scap, 8) +
                  65536;
    return SYMDEL_OK;
}

int symdel_self(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d, void* workspace,
                int64_t workspace_bytes, int32_t* out_i, int32_t* out_j, int32_t* out_dist, int64_t capacity,
                int64_t* n_pairs_host, void* cuda_stream) {
    SeqSetDev A{seqs, offsets, n}, B{nullptr, nullptr, 0};
    return run_pipeline(ctx, A, B, 0, d, workspace, workspace_bytes, out_i, out_j, out_dist, capacity, n_pairs_host,
                        (cudaStream_t)cuda_stream);
}

int symdel_cross(symdel_ctx* ctx, const int8_t* q_seqs, const int64_t* q_offsets, int64_t n_q, const int8_t* r_seqs,
                 const int64_t* r_offsets, int64_t n_r, int d, void* workspace, int64_t workspace_bytes, int32_t* out_i,
                 int32_t* out_j, int32_t* out_dist, int64_t capacity, int64_t* n_pairs_host, void* cuda_stream) {
    SeqSetDev A{q_seqs, q_offsets, n_q}, B{r_seqs, r_offsets, n_r};
    return run_pipeline(ctx, A, B, 1, d, workspace, workspace_bytes, out_i, out_j, out_dist, capacity, n_pairs_host,
                        (cudaStream_t)cuda_stream);
}

int symdel_self_host(symdel_ctx* ctx, const int8_t* seqs_host, const int64_t* offsets_host, int64_t n, int d,
                     int32_t* out_i_host, int32_t* out_j_host, int32_t* out_dist_host, int64_t capacity,
                     int64_t* n_pairs_host) {
    return run_host(ctx, seqs_host, offsets_host, n, nullptr, nullptr, 0, 0, d, out_i_host, out_j_host, out_dist_host,
                    capacity, n_pairs_host);
}

int symdel_cross_host(symdel_ctx* ctx, const int8_t* q_seqs_host, const int64_t* q_offsets_host, int64_t n_q,
                      const int8_t* r_seqs_host, const int64_t* r_offsets_host, int64_t n_r, int d, int32_t* out_i_host,
                      int32_t* out_j_host, int32_t* out_dist_host, int64_t capacity, int64_t* n_pairs_host) {
    return run_host(ctx, q_seqs_host, q_offsets_host, n_q, r_seqs_host, r_offsets_host, n_r, 1, d, out_i_host, out_j_host,
                    out_dist_host, capacity, n_pairs_host);
}

int symdel_overlap_matrix(symdel_ctx* ctx, const int32_t* out_i, const int32_t* out_j, int64_t n_pairs, const int32_t* labels_i,
                          int64_t n_labels_i, const int32_t* labels_j, int64_t n_labels_j, int n_repertoires, int symmetric,
                          int64_t* matrix, void* workspace, int64_t workspace_bytes, void* cuda_stream) {
    if (!ctx || n_pairs < 0 || n_repertoires < 1 || n_repertoires > 4096 || !matrix || !labels_i || !labels_j || !workspace ||
        workspace_bytes < 256 || n_labels_i < 0 || n_labels_j < 0 || (n_pairs > 0 && (!out_i || !out_j)))
        return SYMDEL_E_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaSetDevice(ctx->device));
    u32* err = (u32*)workspace;
    CK(cudaMemsetAsync(err, 0, sizeof(u32), st));
    CK(sd_overlap(out_i, out_j, n_pairs, labels_i, n_labels_i, labels_j, n_labels_j, n_repertoires, symmetric ? 1 : 0, (u64*)matrix, err, st));
    CK(cudaMemcpyAsync(&ctx->h_info->err, err, sizeof(u32), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ctx->h_info->err ? SYMDEL_E_ARG : SYMDEL_OK;
}

// ---- stage-level entry points ------------------------------------------------------------------
int64_t symdel_stage_sort_workspace_bytes(int64_t n) { return align_up(sd_sort_scratch_bytes(std::max<i64>(n, 1), 8)) + 256; }

int symdel_stage_sort_u64(symdel_ctx* ctx, uint64_t* keys, uint64_t* tmp, int64_t n, int begin_bit, int end_bit,
                          void* workspace, int64_t workspace_bytes, void* cuda_stream) {
    if (!ctx || n < 0 || begin_bit < 0 || end_bit > 64 || end_bit < begin_bit || (end_bit - begin_bit) % 8 != 0)
        return SYMDEL_E_ARG;
    if (n >= ((i64)1 << 30)) return SYMDEL_E_TOO_MANY;
    if (n == 0 || end_bit == begin_bit) return SYMDEL_OK;
    if (!keys || !tmp || !workspace) return SYMDEL_E_ARG;
    const int npass = (end_bit - begin_bit) / 8;
    if (workspace_bytes < sd_sort_scratch_bytes(n, npass)) return SYMDEL_E_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaSetDevice(ctx->device));
    CK(sd_sort_prepare(workspace, n, npass, st));
    CK(sd_sort_histogram(keys, n, begin_bit, npass, workspace, st, nullptr));
    CK(sd_sort_hist_scan(workspace, npass, st, nullptr));
    u64* res = nullptr;
    CK(sd_sort_passes(keys, tmp, n, nullptr, begin_bit, npass, ctx->opt_sort_grouping ? 0 : 1, (int)ctx->opt_sort_variant, workspace, st, &res, nullptr));
    if (res != keys) CK(cudaMemcpyAsync(keys, res, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    return SYMDEL_OK;
}

int symdel_stage_generate(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d, int hash_bits,
                          int id_bits, int thinning, uint64_t* records, int64_t records_capacity, int64_t* n_records_host,
                          void* workspace, int64_t workspace_bytes, void* cuda_stream) {
    if (!ctx || !n_records_host || n < 0 || d < 0 || d > SD_D_MAX || hash_bits < 1 || hash_bits + id_bits > 64 || id_bits < 1)
        return SYMDEL_E_ARG;
    *n_records_host = 0;
    if (n == 0) return SYMDEL_OK;
    if (!seqs || !offsets || !records || !workspace) return SYMDEL_E_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaSetDevice(ctx->device));
    Bump ws(workspace, workspace_bytes);
    DevInfo* info = ws.take<DevInfo>(1);
    u32* cnt = ws.take<u32>(n);
    u64* rec_off = ws.take<u64>(n + 1);
    u64* scan_lb = ws.take<u64>(sd_scan_tiles(n) + 1);
    u32* hist = ws.take<u32>(8 * 256);
    if (!ws.ok) return SYMDEL_E_WORKSPACE;
    SeqSetDev A{seqs, offsets, n}, B{nullptr, nullptr, 0};
    CK(cudaMemsetAsync(info, 0, sizeof(DevInfo), st));
    CK(cudaMemsetAsync(hist, 0, 8 * 256 * 4, st));
    CK(sd_prepare(A, d, 0, 0, info, st, nullptr));
    CK(sd_check_residues(A, info, st));
    int rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    Layout lay{};
    lay.n_a = n;
    lay.d = d;
    lay.id_bits = id_bits;
    lay.hash_bits = hash_bits;
    lay.thinning = thinning;
    lay.force_general = ctx->opt_general_gen ? 1 : 0;
    lay.n_chunks = 1;
    const int width = (int)ctx->h_info->maxlen + 1;
    CK(sd_count(A, B, lay, width, cnt, info, st, nullptr));
    CK(sd_scan_counts(cnt, n, rec_off, scan_lb, info, st, nullptr));
    rc = read_info(ctx, info, st);
    if (rc) return rc;
    const i64 N = (i64)ctx->h_info->n_records;
    *n_records_host = N;
    if (N > records_capacity) return SYMDEL_E_CAPACITY;
    CK(sd_generate(A, B, lay, width, rec_off, records, hist, id_bits, 0, info, st, nullptr));
    rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    return SYMDEL_OK;
}

int symdel_stage_generate_fused(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d, int hash_bits, int id_bits,
                                int thinning, int n_chunks, uint64_t chunk_lo, uint64_t chunk_hi, uint64_t* bins, int64_t bin_capacity,
                                uint32_t* bin_counts, int64_t* n_records_host, void* workspace, int64_t workspace_bytes,
                                void* cuda_stream) {
    if (!ctx || !n_records_host || n < 0 || d < 0 || d > SD_D_MAX || hash_bits < 8 || hash_bits + id_bits > 64 || id_bits < 1 ||
        n_chunks < 1 || bin_capacity < 32 || bin_capacity % 32 != 0 || bin_capacity >= ((i64)1 << 30) || n >= ((i64)1 << id_bits))
        return SYMDEL_E_ARG;
    *n_records_host = 0;
    if (!bins || !bin_counts || !workspace) return SYMDEL_E_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemsetAsync(bin_counts, 0, 256 * sizeof(u32), st));
    if (n == 0) {
        CK(cudaStreamSynchronize(st));
        return SYMDEL_OK;
    }
    if (!seqs || !offsets) return SYMDEL_E_ARG;
    Bump ws(workspace, workspace_bytes);
    DevInfo* info = ws.take<DevInfo>(1);
    if (!ws.ok) return SYMDEL_E_WORKSPACE;
    SeqSetDev A{seqs, offsets, n}, B{nullptr, nullptr, 0};
    CK(cudaMemsetAsync(info, 0, sizeof(DevInfo), st));
    CK(sd_prepare(A, d, 0, 0, info, st, nullptr));
    CK(sd_check_residues(A, info, st));
    int rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    Layout lay{};
    lay.n_a = n;
    lay.d = d;
    lay.id_bits = id_bits;
    lay.b_bits = id_bits;
    lay.pair_bits = 2 * id_bits;
    lay.hash_bits = hash_bits;
    lay.sort_bits = 8;
    lay.thinning = thinning;
    lay.force_general = ctx->opt_general_gen ? 1 : 0;
    lay.n_chunks = (u32)n_chunks;
    lay.chunk_lo = n_chunks > 1 ? chunk_lo : 0ull;
    lay.chunk_hi = n_chunks > 1 ? chunk_hi : ~0ull;
    const int width = (int)ctx->h_info->maxlen + 1;
    if (!sd_gen_part_applies(lay, width)) return SYMDEL_E_ARG;
    const double rpr = (double)ctx->h_info->nmax / (double)std::max<i64>((i64)ctx->h_info->residues, 1) / (double)n_chunks;
    CK(sd_gen_part(A, B, lay, width, bins, bin_counts, (u64)bin_capacity, rpr, (double)ctx->h_info->residues / (double)n, 0, -1, 1, info, st, nullptr));
    u32* h_cur = reinterpret_cast<u32*>(ctx->h_info + 1);
    CK(cudaMemcpyAsync(h_cur, bin_counts, 256 * sizeof(u32), cudaMemcpyDeviceToHost, st));
    rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    i64 total = 0;
    for (int i = 0; i < 256; ++i) total += h_cur[i];
    *n_records_host = total;
    return ctx->h_info->part_overflow ? SYMDEL_E_CAPACITY : SYMDEL_OK;
}

int symdel_stage_lev(symdel_ctx* ctx, const int8_t* a_seqs, const int64_t* a_offsets, int64_t n_a, const int8_t* b_seqs,
                     const int64_t* b_offsets, int64_t n_b, const int32_t* ia, const int32_t* ib, int64_t n_pairs,
                     int32_t* dist, void* workspace, int64_t workspace_bytes, void* cuda_stream) {
    if (!ctx || n_pairs < 0 || n_a < 0 || n_b < 0) return SYMDEL_E_ARG;
    if (n_pairs == 0) return SYMDEL_OK;
    if (!a_seqs || !a_offsets || !b_seqs || !b_offsets || !ia || !ib || !dist || !workspace) return SYMDEL_E_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaSetDevice(ctx->device));
    SeqSetDev A{a_seqs, a_offsets, n_a}, B{b_seqs, b_offsets, n_b};
    Bump ws(workspace, workspace_bytes);
    DevInfo* info = ws.take<DevInfo>(1);
    void* slots = ws.take<char>(sd_pack_bytes(n_a + n_b, SD_L_MAX));
    if (!ws.ok) return SYMDEL_E_WORKSPACE;
    CK(cudaMemsetAsync(info, 0, sizeof(DevInfo), st));
    CK(sd_prepare(A, 0, 0, 0, info, st, nullptr));
    CK(sd_prepare(B, 0, 1, 0, info, st, nullptr));
    int rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err) return err_from_flags(ctx->h_info->err);
    const int maxlen = (int)ctx->h_info->maxlen;
    CK(sd_pack(A, B, maxlen, slots, info, st, nullptr));
    CK(sd_lev_pairs(slots, n_a, n_b, maxlen, ia, ib, n_pairs, dist, &info->err, st));
    rc = read_info(ctx, info, st);
    if (rc) return rc;
    if (ctx->h_info->err & SD_ERR_RESIDUE) return SYMDEL_E_RESIDUE;
    return ctx->h_info->err ? SYMDEL_E_ARG : SYMDEL_OK;
}

}  // extern "C"
