/* symdel.h — C ABI of libsymdel: symmetric-deletion (SymDel) Levenshtein neighbour search on one
 * NVIDIA B200 (sm_100a).  arxiv/paper_2403_09010, "Lightning-fast adaptive immune receptor
 * similarity search by symmetric deletion lookup".
 *
 * The operation (App. F.1 steps 0-5; App. F.3): "Given an array
 * {s_i} of AIR sequences and a distance threshold ... return {(i, i', d(s_i, s_i'))}", computed by
 * (1) generating every deletion variant with up to d deletions of every sequence, (2) a sort-merge
 * join of the variants (§I.B), (3) candidate-pair emission and deduplication,
 * (4) exact edit-distance verification on the full sequences.  The two-set form
 * ("for both the query and reference sets"; Fig. 1) is symdel_cross.
 *
 * Result contract
 *   symdel_self : every pair 0 <= i < j < n with lev(s_i, s_j) <= d exactly once, dist = the exact
 *                 unit-cost Levenshtein distance (0..d), sorted ascending by (i, j).
 *   symdel_cross: every (q, r) with lev(query_q, ref_r) <= d exactly once, sorted ascending by (q, r).
 *   Indices are positions in the caller's arrays.  Exact duplicates are legal and reported at
 *   dist 0 (the paper only recommends collapsing them).  Empty sequences are legal.
 *
 * Sequences are CSR: `seqs` int8 residue codes 1..31 (0 is reserved), `offsets` int64[n+1] with
 * offsets[0] == 0, non-decreasing; sequence i is seqs[offsets[i] .. offsets[i+1]).
 *
 * Pointers are DEVICE pointers unless the parameter name ends in `_host`.  The library never
 * allocates or frees caller memory; device entry points never call cudaMalloc (the caller passes a
 * workspace); the *_host entry points stage through a device arena owned by the context.
 * Every function returns SYMDEL_OK (0) or a negative SYMDEL_E_* code; nothing throws or aborts
 * across the ABI.  On error the outputs are unspecified unless stated.  All calls are synchronous
 * with respect to the result: when they return, outputs and *n_pairs_host are final.
 * There is no CPU fallback: without a CUDA device every compute entry point fails with SYMDEL_E_CUDA.
 *
 * Devices and threads.  A context belongs to the device given to symdel_create: every call through it selects
 * that device (cudaSetDevice) and expects device pointers and the stream of that device.  All per-device state
 * of the library (constant hash tables, kernel attributes) is set up by symdel_create for the context's own
 * device, so contexts on several GPUs can coexist in one process.  A context is NOT re-entrant: at most one host
 * thread may be inside a call on a given context at any time (it owns one pinned status block, one stats
 * record and, for the *_host calls, one arena).  Different contexts — on the same or on different devices — may
 * be used from different host threads concurrently; symdel_create / symdel_destroy may be called concurrently.
 * symdel_strerror and symdel_workspace_bytes are pure functions.
 */
#ifndef SYMDEL_H
#define SYMDEL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SYMDEL_API __attribute__((visibility("default")))
#else
#define SYMDEL_API
#endif

#define SYMDEL_D_MAX 4   /* largest distance threshold accepted (the paper benchmarks d <= 5; configs need <= 3) */
#define SYMDEL_L_MAX 64  /* longest sequence accepted = one 64-bit word of the bit-parallel verifier (configs need <= 30) */

enum {
    SYMDEL_OK = 0,
    SYMDEL_E_ARG = -1,       /* null pointer, n < 0, d < 0 or d > SYMDEL_D_MAX, bad option */
    SYMDEL_E_OFFSETS = -2,   /* offsets[0] != 0 or offsets decreasing */
    SYMDEL_E_TOO_LONG = -3,  /* some sequence longer than SYMDEL_L_MAX */
    SYMDEL_E_RESIDUE = -4,   /* residue code outside 1..31 */
    SYMDEL_E_TOO_MANY = -5,  /* n_a + n_b >= 2^30 */
    SYMDEL_E_WORKSPACE = -6, /* workspace too small even at maximum chunking */
    SYMDEL_E_CAPACITY = -7,  /* more result pairs than `capacity`: the first `capacity` pairs (ascending) are valid; *n_pairs_host = the required
                                count — exact, except when a chunked / windowed search had to cut its survivor list (stats.surv_merges > 0
                                and the list exceeded `capacity`): then a lower bound of it, still > capacity */
    SYMDEL_E_CUDA = -8,      /* CUDA error (sticky); code via symdel_last_cuda_error */
    SYMDEL_E_INTERNAL = -9,  /* internal consistency check failed (never expected) */
    SYMDEL_E_STATIC_LIMIT = -10 /* symdel_sort_u64_static: n > SYMDEL_STATIC_SORT_MAX_KEYS (its built-in scratch cannot grow) */
};

typedef struct symdel_ctx symdel_ctx; /* opaque; owns small pinned scratch, stats and (host entry points only) a device arena */

/* Stage counters and timings of the LAST call (Table S1's columns).
 * n_candidates / n_unique depend on the key hash and are not comparable with the paper's. */
typedef struct {
    int64_t n_records;     /* (variant key, id) records generated = distinct (variant, id) tuples */
    int64_t n_candidates;  /* candidate pairs emitted by the join (distinct ids, before dedup) */
    int64_t n_unique;      /* candidates after dedup */
    int64_t n_outputs;     /* verified pairs */
    int64_t n_chunks;      /* key-range chunks used (S5) */
    int64_t n_flushes;     /* candidate-buffer flushes (dedup+verify rounds) */
    int64_t n_launches;    /* kernels launched */
    int32_t hash_bits;     /* hash bits carried per record (64 - id_bits unless narrowed) */
    int32_t id_bits;       /* id bits per record */
    int32_t sort_bits;     /* top hash bits radix-partitioned by S2 (8 per onesweep pass); the join compares the rest */
    int32_t join_general;  /* chunks whose join ran the general (windowed) kernel instead of the fast one */
    float ms_prepare, ms_generate, ms_sort, ms_emit, ms_dedup, ms_verify, ms_total; /* CUDA-event times; 0 unless SYMDEL_OPT_TIMING is set */
    float ms_sort_pass_avg; /* average duration of one onesweep pass over the variant records */
    int64_t sort_pass_records; /* records moved by one such pass */
    int64_t fused_chunks;      /* chunks that went through the fused pipeline (generation + partition in one kernel, bucket join) */
    int64_t join_redo_tiles;   /* join tiles that overflowed the small candidate list and were redone by the large-list kernel */
    int64_t surv_merges;       /* multi-flush searches: times the survivor list was sorted and deduplicated to make room */
    int64_t join_windows;      /* fused pipeline: extra passes of the bucket join (the pairs of a chunk exceeded one candidate window) */
    int64_t query_filter_bits; /* cross-search: 2^bits filter bits per level-1 bin when the query filter ran (0: it did not) */
} symdel_stats;

/* Options (symdel_set_option); defaults in brackets. */
enum {
    SYMDEL_OPT_TIMING = 1,        /* [0] 1: bracket each stage with CUDA events (adds stream syncs at the end only) */
    SYMDEL_OPT_FORCE_CHUNKS = 2,  /* [0] >0: use exactly this many key-range chunks (test hook for S5) */
    SYMDEL_OPT_CAND_CAPACITY = 3, /* [0] >0: cap the candidate buffer at this many pairs (test hook for multi-flush) */
    SYMDEL_OPT_HASH_BITS = 4,     /* [0] 0 = every bit the id leaves free; else 1..63: hash bits kept per record (test hook: a narrow hash makes colliding variants, the result is unchanged) */
    SYMDEL_OPT_NO_THINNING = 5,   /* [0] 1: emit one record per deletion SET instead of per distinct variant (test hook) */
    SYMDEL_OPT_SORT_VARIANT = 6,  /* [0] 0..3: tile shape of the onesweep kernel used by this context (test hook: other tile geometries; results are identical) */
    SYMDEL_OPT_GENERAL_GENERATE = 7, /* [0] 1: use the general (any d, any length) generation kernel even where the d <= 2 fast path applies (test hook) */
    SYMDEL_OPT_SORT_BITS = 8,     /* [0] 0 = automatic; 8..56 (multiple of 8): top hash bits that S2 radix-partitions; 255 = none (one bucket: the join chunks it) */
    SYMDEL_OPT_SORT_STABLE = 9,   /* [0] 1: every S2 pass takes the stable (ties keep input order) tile path (test hook; results are identical) */
    SYMDEL_OPT_SORT_GROUPING = 10,/* [0] 1: symdel_stage_sort_u64 sorts keys only: ties land in arbitrary order (the mode the pipeline uses) */
    SYMDEL_OPT_JOIN_GENERAL = 11, /* [0] 1: always run the general join kernel (windowed output, chunked buckets) instead of trying the fast one first (test hook; results are identical) */
    SYMDEL_OPT_EXACT_PIPELINE = 12, /* [0] 1: never use the fused pipeline (fixed-capacity bins); always count, scan, generate, onesweep-partition on exact histograms, windowed join (the path the fused one falls back to when a bin overflows; results are identical) */
    SYMDEL_OPT_PREFIX_LEN = 13,   /* [0] P > 0: prefix-truncated candidate generation (App. B; XTNeighbor uses 18): deletion variants are generated from the first P residues of every sequence, verification stays on the whole sequences.  Exact for P > d (calls with P <= d return SYMDEL_E_ARG); fewer records, more candidates */
    SYMDEL_OPT_METRIC = 14,       /* [0] 0: Levenshtein distance (the paper's metric).  1: Hamming distance (Fig. S3 A/C): only pairs of EQUAL length with <= d mismatching positions are returned, dist = the mismatch count; candidates come from the same deletion-variant join (hamming <= d implies lev <= d) */
    SYMDEL_OPT_SURV_CAPACITY = 15, /* [0] >0: size of the survivor list of multi-flush searches in pairs (test hook; never below capacity + 4096: a candidate window whose survivors do not fit behind the list is verified in slices, the list being sorted, deduplicated and cut to its smallest `capacity` pairs in between) */
    SYMDEL_OPT_CAND_FILTER = 16, /* [0] duplicate suppression before the candidate sort (a best-effort hash set of pair ids): 0 = automatic (on when the candidates are many but few per record), 1 = always, 2 = never (test hook; results are identical) */
    SYMDEL_OPT_NO_QUERY_FILTER = 17, /* [0] 1: cross-search never drops reference records through the query filter (test hook: same result) */
    SYMDEL_OPT_FLUSH_PER_CHUNK = 18 /* [0] 1: a chunked search deduplicates and verifies its candidates after EVERY key-range chunk instead of letting the chunks append to one candidate window that is flushed when it fills or after the last chunk (test hook; results are identical) */
};

/* ---- context ------------------------------------------------------------------------------- */
SYMDEL_API int symdel_create(symdel_ctx** ctx, int device);  /* selects `device`; SYMDEL_E_CUDA if there is none or it is not a B200 (compute capability 10.0, 148 SMs, 227 KB shared memory per block: the kernels are built and sized for exactly that) */
SYMDEL_API void symdel_destroy(symdel_ctx* ctx);
SYMDEL_API int symdel_set_option(symdel_ctx* ctx, int option, int64_t value);
SYMDEL_API int symdel_get_stats(const symdel_ctx* ctx, symdel_stats* stats_host);
SYMDEL_API int symdel_last_cuda_error(const symdel_ctx* ctx); /* cudaError_t of the last SYMDEL_E_CUDA, else 0 */
SYMDEL_API const char* symdel_strerror(int code);             /* static string */

/* Recommended workspace size for an un-chunked run.  n_b = 0 and residues_b = 0 for self-search.
 * max_len = longest sequence (<= SYMDEL_L_MAX); capacity = the output capacity that will be passed.
 * Any workspace >= the minimum the library needs works: a smaller one makes symdel_* split the key
 * space into chunks (S5).  Pure host arithmetic. */
SYMDEL_API int symdel_workspace_bytes(int64_t n_a, int64_t residues_a, int64_t n_b, int64_t residues_b, int max_len, int d,
                           int64_t capacity, int64_t* bytes_host);

/* ---- the hot path, device-resident inputs and outputs ---------------------------------------
 * out_i/out_j/out_dist: caller-owned device arrays of `capacity` int32 each.
 * workspace: caller-owned device memory, 256-byte aligned, contents destroyed.
 * cuda_stream: a cudaStream_t (may be NULL = default stream); all work is issued on it. */
SYMDEL_API int symdel_self(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d, void* workspace,
                int64_t workspace_bytes, int32_t* out_i, int32_t* out_j, int32_t* out_dist, int64_t capacity,
                int64_t* n_pairs_host, void* cuda_stream);

SYMDEL_API int symdel_cross(symdel_ctx* ctx, const int8_t* q_seqs, const int64_t* q_offsets, int64_t n_q, const int8_t* r_seqs,
                 const int64_t* r_offsets, int64_t n_r, int d, void* workspace, int64_t workspace_bytes,
                 int32_t* out_i, int32_t* out_j, int32_t* out_dist, int64_t capacity, int64_t* n_pairs_host,
                 void* cuda_stream);

/* ---- the same calls with HOST buffers (inputs copied host->device and results device->host
 * inside the call; pinned host memory makes the copies asynchronous).  The offsets are sent first (input
 * validation and sizing need nothing else), a large self-search sends the residues in slices and generates
 * variants of a slice while the next is on its way.  The device arena is sized from an estimate of the record
 * count; a low estimate only makes the search run in key-range chunks. ------------------------------------- */
SYMDEL_API int symdel_self_host(symdel_ctx* ctx, const int8_t* seqs_host, const int64_t* offsets_host, int64_t n, int d,
                     int32_t* out_i_host, int32_t* out_j_host, int32_t* out_dist_host, int64_t capacity,
                     int64_t* n_pairs_host);

SYMDEL_API int symdel_cross_host(symdel_ctx* ctx, const int8_t* q_seqs_host, const int64_t* q_offsets_host, int64_t n_q,
                      const int8_t* r_seqs_host, const int64_t* r_offsets_host, int64_t n_r, int d,
                      int32_t* out_i_host, int32_t* out_j_host, int32_t* out_dist_host, int64_t capacity,
                      int64_t* n_pairs_host);

/* NEXT-4: "aggregates an M x M overlap matrix from identified neighbor pairs, where each entry
 * contains the number of neighbors between two repertoires".  out_i/out_j: the n_pairs result pairs of a
 * symdel_self / symdel_cross call (device); labels_i[x] / labels_j[y] in [0, n_repertoires): the repertoire of
 * the sequence behind first / second pair component (device; the same array for a self-search);
 * matrix: device int64[M * M], row-major, OVERWRITTEN: matrix[p][q] = #pairs with labels (p, q).  symmetric = 1
 * (self-search, reading A-18): a pair with labels p != q also counts in [q][p]; within-repertoire pairs count once
 * on the diagonal.  n_labels_i / n_labels_j: lengths of the label arrays (= the sizes of the searched sets).
 * workspace: >= 256 device bytes.  Synchronises the stream.  SYMDEL_E_ARG if a pair index lies outside its label
 * array or a label outside [0, n_repertoires) (the matrix is then unspecified; nothing is read out of bounds), or
 * if n_repertoires is outside 1..4096. */
SYMDEL_API int symdel_overlap_matrix(symdel_ctx* ctx, const int32_t* out_i, const int32_t* out_j, int64_t n_pairs,
                          const int32_t* labels_i, int64_t n_labels_i, const int32_t* labels_j, int64_t n_labels_j,
                          int n_repertoires, int symmetric, int64_t* matrix, void* workspace, int64_t workspace_bytes,
                          void* cuda_stream);

/* ---- stage-level entry points (kernel parity tests and micro-benchmarks) ---------------------
 * S2/K2: stable LSD radix sort of n 64-bit keys on bits [begin_bit, end_bit) (end - begin a
 *   multiple of 8).  keys and tmp: device arrays of n; the sorted result is left in `keys`.
 *   workspace: device scratch of at least symdel_stage_sort_workspace_bytes(n) bytes. */
SYMDEL_API int64_t symdel_stage_sort_workspace_bytes(int64_t n);
SYMDEL_API int symdel_stage_sort_u64(symdel_ctx* ctx, uint64_t* keys, uint64_t* tmp, int64_t n, int begin_bit, int end_bit,
                          void* workspace, int64_t workspace_bytes, void* cuda_stream);

/* S1/K1: (key, id) records of one sequence set, unsorted, in id order: records[t] =
 *   (hash >> (64 - hash_bits)) << id_bits | id.  Returns the count through *n_records_host.
 *   thinning = 1: one record per distinct variant (leftmost embedding); 0: one per deletion set. */
SYMDEL_API int symdel_stage_generate(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d, int hash_bits,
                          int id_bits, int thinning, uint64_t* records, int64_t records_capacity,
                          int64_t* n_records_host, void* workspace, int64_t workspace_bytes, void* cuda_stream);

/* S1+S2 fused (the generator of the default pipeline: k_gen2_part for d <= 3 and sequences of <= 32 residues, else
 *   k_generate_part; SYMDEL_OPT_GENERAL_GENERATE forces the latter): the same records as symdel_stage_generate, but
 *   pushed straight into 256 bins by the top 8 bits of their hash field — bins[b * bin_capacity + t], t < bin_counts[b]
 *   (device u32[256], overwritten), in no particular order inside a bin.  bin_capacity: a multiple of 32, < 2^30.
 *   n_chunks > 1 selects the key-range-chunk instance (S5): only records whose position (variant length << 32 | hash
 *   fraction) lies in [chunk_lo, chunk_hi) are made; n_chunks == 1 ignores the two bounds.  *n_records_host = records
 *   pushed.  SYMDEL_E_CAPACITY: some bin was full (records beyond bin_capacity were dropped; the pipeline then falls back to
 *   its exact form).  workspace: >= 4096 device bytes.  n must be < 2^id_bits and hash_bits >= 8. */
SYMDEL_API int symdel_stage_generate_fused(symdel_ctx* ctx, const int8_t* seqs, const int64_t* offsets, int64_t n, int d,
                                int hash_bits, int id_bits, int thinning, int n_chunks, uint64_t chunk_lo, uint64_t chunk_hi,
                                uint64_t* bins, int64_t bin_capacity, uint32_t* bin_counts, int64_t* n_records_host,
                                void* workspace, int64_t workspace_bytes, void* cuda_stream);

/* S4/K6: dist[t] = lev(a_{ia[t]}, b_{ib[t]}) by the bit-parallel verifier, for n_pairs index pairs.
 *   workspace: device scratch of at least 512 + 48 * (n_a + n_b) bytes (the packed bit-plane table).
 *   An index outside [0, n_a) / [0, n_b) gives dist[t] = -1 and the call returns SYMDEL_E_ARG. */
SYMDEL_API int symdel_stage_lev(symdel_ctx* ctx, const int8_t* a_seqs, const int64_t* a_offsets, int64_t n_a,
                     const int8_t* b_seqs, const int64_t* b_offsets, int64_t n_b, const int32_t* ia,
                     const int32_t* ib, int64_t n_pairs, int32_t* dist, void* workspace, int64_t workspace_bytes,
                     void* cuda_stream);

/* ---- a sort that allocates nothing and needs no workspace --------------------------------------------------------
 * symdel_sort_u64_static = symdel_stage_sort_u64 (stable LSD radix sort of n 64-bit keys on bits [begin_bit, end_bit),
 * end - begin a multiple of 8, result left in `keys`; the sort of the sort-merge join) for callers
 * that cannot give the library any device memory beyond the data itself: plug-ins inside an application whose pool
 * already owns the whole GPU (cudaMalloc fails there), service loops where cudaMalloc / cudaFree are banned because they
 * can synchronise the device, error paths that run after an out-of-memory.  The caller passes only `keys` (device,
 * n x uint64, read and overwritten).  The ping-pong buffer and the status words sit in a __device__ array inside
 * libsymdel.so: SYMDEL_STATIC_SORT_SCRATCH_BYTES (11 MiB) of every GPU that loads the library, held until the process
 * exits — hence the limit n <= SYMDEL_STATIC_SORT_MAX_KEYS (2^20); a larger n returns SYMDEL_E_STATIC_LIMIT and
 * touches nothing.  The call needs no symdel_ctx (creating one allocates) and performs no cudaMalloc / cudaFree or
 * any other allocating call; it selects `device` (cudaSetDevice), issues its work on `cuda_stream` (a cudaStream_t of
 * that device, NULL = default stream) and returns after synchronising that stream, like every call of this header.
 *   - First call on a device: looks up the array's device address and sets the sort kernels' shared-memory limit.
 *     Make that call before any stream capture begins; later calls on the device skip the set-up.
 *   - One array per GPU, shared by all calls and never reset between them: each call clears the words that must start
 *     at zero on `cuda_stream` before its kernels.  Calls on the same device whose GPU work may overlap (other streams,
 *     other host threads) race on the array — the result is undefined; serialise them.
 * Errors: SYMDEL_E_ARG (bad bit range, n < 0, null keys, device outside 0..63), SYMDEL_E_STATIC_LIMIT, SYMDEL_E_CUDA
 * (no such device or a CUDA call failed; cudaGetLastError has the code — there is no context to keep it). */
#define SYMDEL_STATIC_SORT_MAX_KEYS 1048576
#define SYMDEL_STATIC_SORT_SCRATCH_BYTES 11534336 /* 8 MiB ping-pong keys + 3 MiB histograms / tickets / status words */
SYMDEL_API int symdel_sort_u64_static(int device, uint64_t* keys, int64_t n, int begin_bit, int end_bit, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* SYMDEL_H */
