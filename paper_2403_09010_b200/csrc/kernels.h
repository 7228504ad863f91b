// kernels.h — internal host-side launch interface between the pipeline (symdel_api.cu) and the
// kernel translation units.  Not part of the public ABI (that is include/symdel.h).
#pragma once
#include <algorithm>
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"


// One CSR sequence set on the device.
struct SeqSetDev {
    const int8_t* seqs;
    const i64* off;
    i64 n;
};

// Everything the record/pair layout depends on, fixed per call.
struct Layout {
    i64 n_a, n_b;      // self: n_b == 0.  Global id = index in A, or n_a + index in B.
    int cross;         // 1: emit only (A, B) combinations
    int d;
    int id_bits;       // 2^id_bits > n_a + n_b
    int hash_bits;     // hash bits kept per record: the record is (hash >> (64 - hash_bits)) << id_bits | id
    int sort_bits;     // multiple of 8, <= hash_bits: the top bits of the hash field that S2 radix-partitions
    int b_bits;        // bits of the second pair component (self: id_bits; cross: bits of n_b)
    int pair_bits;     // a_bits + b_bits
    int thinning;
    int prefix;         // > 0: variants come from the first `prefix` residues of every sequence (App. B)
    int metric;         // 0: Levenshtein; 1: Hamming (equal lengths only, mismatch count)
    int force_general;  // test hook: never take the d <= 2 fast generation path
    u32 n_chunks, chunk;
    u64 chunk_lo, chunk_hi;  // S5: this chunk holds the records with chunk_lo <= (variant length << 32 | hash fraction) < chunk_hi
};

// ---- radix_sort.cu ------------------------------------------------------------------------------
i64 sd_sort_tiles(i64 n);
int sd_sort_variants();           // number of selectable tile shapes of k_onesweep
cudaError_t sd_sort_setup();      // per-device setup (function attributes); symdel_create
i64 sd_sort_scratch_bytes(i64 n, int npass);
cudaError_t sd_sort_prepare(void* scratch, i64 n, int npass, cudaStream_t st);
u32* sd_sort_hist_ptr(void* scratch);
cudaError_t sd_sort_histogram(const u64* keys, i64 n, int begin_bit, int npass, void* scratch, cudaStream_t st,
                              i64* launches);
cudaError_t sd_sort_hist_scan(void* scratch, int npass, cudaStream_t st, i64* launches);
// n_dev != nullptr: the key count is *n_dev (device); n is an upper bound that sizes the grids and the scratch
cudaError_t sd_sort_passes(u64* keys, u64* tmp, i64 n, const u64* n_dev, int begin_bit, int npass, int stable, int variant,
                           void* scratch, cudaStream_t st, u64** result, i64* launches);
// S3b duplicate suppression before the sort: keeps the candidates a best-effort hash set has not seen yet, compacts
// them into out[0 .. *n_out) and accumulates their digit histograms (bits [0, 8 * npass)) into `scratch`
cudaError_t sd_cand_filter(const u64* cand, i64 n, void* table, int table_bits, u64* out, u64* n_out, int npass, void* scratch,
                           cudaStream_t st, i64* launches);

// level-2 partition of the fused pipeline: bins (256 x cap1) -> buckets ((256 << b2) x cap2)
#define SD_FBITS_MAX 19  // query filter: at most 2^19 bits (64 KB) per level-1 bin (config 4 with 17 / 18 / 19 bits: 6.4 / 5.8 / 5.5 ms: fewer survivors beat more resident blocks)
// bitmap != nullptr: the query filter of a cross-search (radix_sort.cu, k_bin_bitmap): 256 bitmaps of 2^fbits bits built by
// sd_bin_bitmap from the first cnt_a[bin] records of every bin; fshift = position of the fbits hash bits below the bin digit
cudaError_t sd_bin_bitmap(const u64* bins, const u32* cnt_a, i64 cap1, u32* bitmap, int fbits, int fshift, cudaStream_t st, i64* launches);
cudaError_t sd_part2(const u64* bins, const u32* cnt1, i64 cap1, u64* buckets, u32* cnt2, i64 cap2, int b2, int shift,
                     int counts_cleared, const u32* bitmap, const u32* cnt_a, int fbits, int fshift, DevInfo* info, cudaStream_t st,
                     i64* launches);

// ---- generate.cu --------------------------------------------------------------------------------
cudaError_t sd_generate_setup();  // per-device setup: the __constant__ tables and function attributes; symdel_create
// validates the offsets and lengths (info->err), accumulates nmax / residues / maxlen; never reads `seqs`
cudaError_t sd_prepare(SeqSetDev s, int d, int is_b, int prefix, DevInfo* info, cudaStream_t st, i64* launches);
// residue codes in 1..31 (info->err |= SD_ERR_RESIDUE); a no-op unless sd_prepare left info->err == 0
cudaError_t sd_check_residues(SeqSetDev s, DevInfo* info, cudaStream_t st);
// count pass: cnt[gid] = number of records sequence gid contributes (u32 per sequence)
cudaError_t sd_count(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, u32* cnt, DevInfo* info, cudaStream_t st,
                     i64* launches);
// exclusive scan cnt -> rec_off[n+1]; total also stored in info->n_records.  lb_status: n/2048+1 u64, zeroed here.
i64 sd_scan_tiles(i64 n);
cudaError_t sd_scan_counts(const u32* cnt, i64 n, u64* rec_off, u64* lb_status, DevInfo* info, cudaStream_t st,
                           i64* launches);
// generation pass: writes records at rec_off[gid].., accumulates the histograms of the npass 8-bit
// digits starting at bit hist_bit of the record into ghist
cudaError_t sd_generate(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, const u64* rec_off, u64* records,
                        u32* ghist, int hist_bit, int npass, DevInfo* info, cudaStream_t st, i64* launches);

// Fused fast path: generation + level-1 partition into 256 bins of cap1 records (cur: 256 cursors =
// the bin counts afterwards).  info->part_overflow != 0: a bin was full, redo with the exact pipeline.
bool sd_gen_part_applies(const Layout& lay, int width);
// records_per_residue = (deletion sets of this chunk) / (residues): sizes the generation rounds
// task_end == -2 / -3: set A only / set B only (the later launch appends: pass cursors_cleared).
// [task_begin, task_end): the warp tasks (groups of 32 consecutive sequences, A then B) of this launch; task_end < 0 = all.
// Slices (sd_gen_part_sliceable only) append to the same bins: the launch starting at task 0 clears the cursors (unless the
// caller has: cursors_cleared).
bool sd_gen_part_sliceable(const Layout& lay, int width);
cudaError_t sd_gen_part(SeqSetDev a, SeqSetDev b, const Layout& lay, int width, u64* bins, u32* cur, u64 cap1,
                        double records_per_residue, double avg_len, i64 task_begin, i64 task_end, int cursors_cleared, DevInfo* info,
                        cudaStream_t st, i64* launches);

// ---- join.cu ------------------------------------------------------------------------------------
i64 sd_join_tiles(i64 n_records);
cudaError_t sd_join_setup();  // per-device setup (function attributes); symdel_create
// records: partitioned on the top lay.sort_bits bits of the hash field.  Emits the candidate pairs of
// the records whose first flat pair index lies in [win_lo, win_hi) to cand[index - win_lo] (cand_cap
// physical slots: the window plus slack for the last record's overhang); info->win_end = end of what
// was written.  first_round = 1: numbers the pairs (tile_prefix[2 * tiles], info->n_cand = total);
// later rounds reuse the numbering.
cudaError_t sd_join(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 cand_cap, u64 win_lo, u64 win_hi,
                    int first_round, u64* tile_prefix, DevInfo* info, cudaStream_t st, i64* launches);

// Fast path of the join (one window of `window` slots, arbitrary candidate order).  sd_join_fast runs the
// small-list kernel over all tiles; tiles whose list overflowed are left in redo[0 .. info->join_redo)
// (redo: one u32 per tile) for sd_join_fast_redo.  info->n_cand = number of pairs; info->join_fallback != 0:
// redo the whole join with sd_join (the pairs exceed `window`, or a tile overflowed the large list too).
cudaError_t sd_join_fast(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 window, u32* redo,
                         DevInfo* info, cudaStream_t st, i64* launches);
cudaError_t sd_join_fast_redo(const u64* records, i64 n_records, const Layout& lay, u64* cand, u64 window, const u32* redo,
                              u32 n_redo, DevInfo* info, cudaStream_t st, i64* launches);

// Bucket join of the fused pipeline (see join.cu): one block per bucket (regions of `cap` <= sd_join_bkt_max_cap()
// records).  Clears and fills info->n_cand; info->join_fallback != 0: the pairs did not fit `window`:
// cand[0 .. min(n_cand, ~info->nofit_inv)) holds the pairs of the buckets that fit; the others are marked open (bit 31 of their
// count) and a further call with first_pass = 0 joins exactly those.
int sd_join_bkt_max_cap();
int sd_join_bkt_link_bits(u32 cap);  // bits on top of a record that must be constant within a bucket
cudaError_t sd_join_bkt(const u64* buckets, u32* cnt, u32 cap, u32 nbuckets, const Layout& lay, u64* cand, u64 window,
                        int first_pass, int info_fresh, int prefer_small, int append, DevInfo* info, cudaStream_t st, i64* launches);
// (append = 1: info->n_cand is NOT cleared — the window already holds that many pairs and this launch claims behind them)

// ---- verify.cu ----------------------------------------------------------------------------------
i64 sd_verify_tiles(i64 n);
// packed bit-plane table of all sequences (A then B): 32 B (maxlen <= 32) or 48 B per sequence
i64 sd_pack_bytes(i64 n_total, int maxlen);
// (also range-checks every residue code: info->err |= SD_ERR_RESIDUE; call only after the offsets were found valid)
cudaError_t sd_pack(SeqSetDev a, SeqSetDev b, int maxlen, void* slots, DevInfo* info, cudaStream_t st, i64* launches);
// cand sorted ascending.  Drops repeats and a == b (self), computes lev, keeps <= d, appends
// (pair << 3 | dist) in order to surv[surv_base + ...]; info->n_surv = total; info->n_unique += unique.
// (n_dev != nullptr: the candidate count is *n_dev, n_cand an upper bound that sizes the grid)
cudaError_t sd_verify(const u64* cand, i64 n_cand, const u64* n_dev, const void* slots, const Layout& lay, int maxlen, u64* surv,
                      u64 surv_base, u64 surv_capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches);
// the same when this is known to be the ONLY flush of the search: survivors go straight to the SoA outputs
cudaError_t sd_verify_direct(const u64* cand, i64 n_cand, const u64* n_dev, const void* slots, const Layout& lay, int maxlen, i32* out_i,
                             i32* out_j, i32* out_dist, i64 capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches);
// surv sorted ascending (and unique unless dedup = 1).  Unpacks to SoA outputs, first `capacity`
// only; info->n_out = total.  packed_out != nullptr: writes the kept words to packed_out instead (the merge of
// the survivor list between flushes).
cudaError_t sd_finalize(const u64* surv, i64 n_surv, const Layout& lay, int dedup, i32* out_i, i32* out_j, i32* out_dist,
                        u64* packed_out, i64 capacity, u64* lb_status, DevInfo* info, cudaStream_t st, i64* launches);
// plain distances for index pairs (stage test); slots = sd_pack of (A, B)
// (an index outside [0, n_a) / [0, n_b): dist = -1 and SD_ERR_INTERNAL in *err)
cudaError_t sd_lev_pairs(const void* slots, i64 n_a, i64 n_b, int maxlen, const i32* ia, const i32* ib, i64 n_pairs, i32* dist,
                         u32* err, cudaStream_t st);
// NEXT-4: M x M overlap matrix of the output pairs under per-sequence repertoire labels
cudaError_t sd_overlap(const i32* pi, const i32* pj, i64 n, const i32* lab_i, i64 n_i, const i32* lab_j, i64 n_j, int M,
                       int symmetric, u64* matrix, u32* err, cudaStream_t st);
