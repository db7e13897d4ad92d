/* barracuda_b200.h -- C-ABI boundary of the B200-native inexact backward search.
 *
 * What the library computes: for every read of a batch and for both strands, the set of
 * suffix-array intervals [k,l] of every reference substring that aligns to the query within the
 * difference budgets (mismatches + gap opens + gap extensions <= z, a 5' seed with its own limit),
 * deduplicated, sorted, with the minimum difference count per interval.
 *
 * Where the paper defines the operations (PAPER.md = /root/reference/PAPER.md, a prose-only note):
 *   - index wholly resident in GPU memory:                 PAPER.md:64 (sec. 2), :41, :86 (sec. 3.4)
 *   - two pointers k,l updated per base from the index, l-k+1 = number of matches,
 *     crossing = absent:                                   PAPER.md:62 (sec. 2)
 *   - "carefully back up its search and start trying out alternatives" (inexact search):
 *                                                          PAPER.md:62
 *   - hundreds of thousands of reads per launch:
 *   - "zero or more possible alignments" per read:         PAPER.md:100 (sec. 3.7)
 *   - coordinates are needed by the next step (sampe):
 * Everything the paper leaves open (difference model, gap rules, seed, strands, $ handling,
 * limits) is fixed in DESIGN.md "Readings of the paper" (= SURVEY.md 8c, C1..C7).
 *
 * Conventions
 *   - Every function returns BC_OK (0) or a negative bc_status; nothing throws, aborts or prints.
 *   - The library allocates NO device memory: the caller (PyTorch in this repo) owns every device
 *     buffer; sizes come from the *_bytes calls.  "host" / "device" is stated per pointer.
 *   - Host inputs are borrowed for the duration of the call only.
 *   - All work is enqueued on the given CUDA stream (a cudaStream_t passed as void*, NULL = legacy
 *     default stream).  bc_index_upload, bc_align_batch and bc_locate synchronise that stream
 *     before returning, so status codes are final.
 *   - Deterministic: same inputs -> byte-identical outputs whatever the scheduling.
 *   - One bc_index may be used from one host thread at a time.  No CPU fallback exists.
 *   - Alphabet A,C,G,T = 0..3; N (reads only) is flagged in a separate mask; complement = 3-c.
 */
#ifndef BARRACUDA_B200_H
#define BARRACUDA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BC_OK = 0,
    BC_E_INVAL = -1,       /* bad argument (NULL, len 0 or > 256, z > 255, negative option, n >= 2^32-1, ...) */
    BC_E_NOMEM = -2,       /* a caller-provided buffer (d_mem, workspace) is smaller than *_bytes said */
    BC_E_CUDA = -3,        /* a CUDA runtime call or kernel failed */
    BC_E_OVERFLOW = -4,    /* raw-hit arena or hits_capacity too small; see bc_result.n_hits_needed */
    BC_E_UNSUPPORTED = -5
} bc_status;

#define BC_MAX_READ_LEN 256

/* One BWT.  X = T$, '$' smallest; SA = suffix array of X (n+1 rows, SA[0] = n);
 * B[j] = X[SA[j]-1]; B[primary] = '$'.  HOST memory. */
typedef struct {
    uint64_t n;               /* |T|, 1 <= n < 2^32-1 */
    uint64_t primary;         /* row whose BWT symbol is '$' (SA[primary] = 0) */
    const uint64_t *bwt2;     /* n symbols, '$' removed, 2 bits each: symbol j at bits 2*(j%32) of word j/32 */
    uint32_t occ_interval;    /* multiple of 32 */
    const uint32_t *occ;      /* [n/occ_interval + 1][4]: occurrences of A,C,G,T before symbol t*occ_interval */
    uint64_t C[5];            /* C[c] = #{t : T[t] < c}; C[4] = n */
} bc_bwt_host;

/* fwd = BWT of T; rev = BWT of reverse(T) (not complemented); sa[t] = SA_fwd[t*sa_interval],
 * t = 0 .. n/sa_interval (rows of the full n+1-row suffix array).  HOST memory. */
typedef struct {
    bc_bwt_host fwd, rev;
    uint32_t sa_interval;     /* >= 1 */
    const uint32_t *sa;
} bc_index_host;

/* Search options: d = mismatches + gap opens + gap extensions <= z; totals
 * n_go <= max_gap_open, n_ge <= max_gap_ext; seed = first seed_len bases of the read (5' end),
 * enabled iff 0 < seed_len < len, differences inside it <= seed_z; a gap column needs
 * >= indel_end_skip read bases on either side. */
typedef struct {
    int32_t z, max_gap_open, max_gap_ext, seed_len, seed_z, indel_end_skip;
} bc_opts;

/* A batch of reads.  DEVICE memory, borrowed. */
typedef struct {
    const uint32_t *bases2;   /* base i of the stream at bits 2*(i%16) of word i/16 (N stored as 0) */
    const uint32_t *nmask;    /* bit i%32 of word i/32 set iff base i is N; NULL = no N anywhere */
    const uint64_t *off;      /* [n_reads] first base of read r in the stream */
    const uint16_t *len;      /* [n_reads] 1..BC_MAX_READ_LEN */
    uint32_t n_reads;
    uint32_t max_len;         /* caller-declared upper bound of len[] (sizes the per-query rows of the
                                 workspace); a read longer than it -> BC_E_INVAL */
} bc_reads;

typedef struct { uint32_t k, l; uint8_t d, strand; uint16_t zero; } bc_hit;   /* 12 bytes */

/* Output, DEVICE memory, caller-owned.  For read r the hits are hits[hit_offsets[r] ..
 * hit_offsets[r+1]): strand 0 (query = read) first, then strand 1 (query = revcomp(read)), each
 * sorted by (k,l); [k,l] are rows of the FORWARD suffix array for both strands. */
typedef struct {
    uint64_t *hit_offsets;    /* [n_reads+1] */
    bc_hit *hits;
    uint64_t hits_capacity;   /* in hits */
    uint64_t *n_hits_needed;  /* [2]: [0] = total hits after dedup, [1] = raw (pre-dedup) records the
                                 search produced.  Both valid on BC_E_OVERFLOW unless the raw arena
                                 itself overflowed, in which case only [1] is (grow the workspace). */
} bc_result;

typedef struct bc_index bc_index;   /* opaque handle (host object holding device pointers) */

/* Bytes of device memory bc_index_upload needs for this index (lines of both BWTs, SA sample,
 * staging for the transport arrays). */
int bc_index_device_bytes(const bc_index_host *h, size_t *bytes);

/* Copies the transport arrays to the device and re-lays them out (kernel) into 32-byte blocks of 64
 * symbols, two per 64-byte line: {uint32 cnt[4]; uint32 lo[2]; uint32 hi[2]} = occurrences of A,C,G,T
 * before symbol 64*i and the two bit-planes of symbols 64*i .. 64*i+63, so that one rank query O(.,j)
 * for all four symbols is ONE aligned 256-bit load inside one 64-byte line (north_star).
 * d_mem: DEVICE, 256-byte aligned, >= bc_index_device_bytes, owned by the caller and must outlive
 * the handle. */
int bc_index_upload(const bc_index_host *h, void *d_mem, size_t d_bytes, void *cuda_stream, bc_index **out);

/* Frees the handle only; d_mem stays the caller's. */
int bc_index_free(bc_index *ix);

/* Workspace bytes for a batch: fixed part (prepared queries with their D[] bounds, the per-warp
 * overflow area of the search kernel's state rings -- sized for the geometry set on the index when
 * this is called -- and counters) + a raw-hit arena of raw_hits_per_read * n_reads records (0 = default 16). */
int bc_align_workspace_bytes(const bc_index *ix, uint32_t n_reads, uint32_t max_len, const bc_opts *o,
                             uint32_t raw_hits_per_read, size_t *bytes);

/* The hot path: D[] bounds, inexact search of both strands 5'->3', hit emission,
 * per-read sort + dedup -> CSR.  d_workspace: DEVICE, 256-byte aligned; whatever ws_bytes exceeds
 * the fixed part becomes the raw-hit arena.  Returns BC_E_OVERFLOW (never truncates) when the arena
 * or hits_capacity is too small; the output is then undefined except n_hits_needed. */
int bc_align_batch(const bc_index *ix, const bc_reads *reads, const bc_opts *o, bc_result *res,
                   void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* Best-stratum mode (the early-terminating behaviour of production short-read
 * aligners, "85 % match uniquely"): per read, exactly the hits of bc_align_batch whose
 * d <= min(d_min + stratum_plus, z), d_min = the read's smallest d over both strands; reads without
 * a hit within z stay empty.  Computed INSIDE the persistent search kernel: every read is searched with its own
 * budget 0, 1, 2, ... by the warp that drew it until its first hits appear (they all have d = d_min), then once
 * more with min(d_min + stratum_plus, z); one launch of the hot path, so well-matching reads never pay for the deep
 * budgets and nothing waits on the host.  Same buffers, layout, ordering and status codes as bc_align_batch (the
 * raw-hit arena also holds the first-hit round's records, which the final round repeats);
 * bc_last_stats[15] = largest per-read budget searched + 1.  bc_align_best_workspace_bytes = bc_align_workspace_bytes
 * (hits_capacity is ignored; kept for source compatibility). */
int bc_align_best_workspace_bytes(const bc_index *ix, uint32_t n_reads, uint32_t max_len, const bc_opts *o,
                                  uint32_t raw_hits_per_read, uint64_t hits_capacity, size_t *bytes);
int bc_align_batch_best(const bc_index *ix, const bc_reads *reads, const bc_opts *o, int32_t stratum_plus,
                        bc_result *res, void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* Pairing of the two ends of a fragment by plausible distance (SURVEY 8f NEXT-1; PAPER.md:37, :39,
 * :104: the `sampe` step).  Input: the DEVICE CSR result of bc_align_batch / bc_align_batch_best for
 * a batch whose reads 2i, 2i+1 are the ends of pair i, and the reads' len[] (DEVICE).  Every hit with
 * <= max_occ occurrences is located into placements (pos, strand, d); a proper pair = one end on
 * strand 0 at pf, the other on strand 1 at pr >= pf, pr + len(reverse end) - pf in [min_frag, max_frag].
 * Output (DEVICE, caller-owned): per pair the records sorted by (pos1, pos2, strand1), one per key
 * with the smallest d1+d2 (then d1); pos1/d1/strand1 belong to read 2i, pos2/d2 to read 2i+1.
 * n_needed[4] (DEVICE): pairs after dedup, candidate pairs, placements, hits skipped for max_occ --
 * on BC_E_OVERFLOW they say what max_placements / max_raw_pairs / pairs_capacity must be. */
typedef struct { uint32_t min_frag, max_frag, max_occ; } bc_pair_opts;
typedef struct { uint32_t pos1, pos2, frag; uint8_t d1, d2, strand1, zero; } bc_pair;   /* 16 bytes */
typedef struct { uint64_t *pair_offsets; bc_pair *pairs; uint64_t pairs_capacity; uint64_t *n_needed; } bc_pair_result;
int bc_pair_workspace_bytes(uint32_t n_reads, uint64_t max_placements, uint64_t max_raw_pairs, size_t *bytes);
int bc_pair_batch(const bc_index *ix, const uint64_t *d_hit_offsets, const bc_hit *d_hits, const uint16_t *d_len,
                  uint32_t n_reads, const bc_pair_opts *o, uint64_t max_placements, uint64_t max_raw_pairs,
                  bc_pair_result *res, void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* SA-interval row -> text coordinate: pos[i] = SA_fwd[rows[i]] by LF-walk to
 * a sampled row.  d_rows, d_pos: DEVICE.  rows[i] must be in [0, n]. */
int bc_locate(const bc_index *ix, const uint32_t *d_rows, uint64_t n_rows, uint32_t *d_pos, void *cuda_stream);

/* Device-side counters of the last bc_align_batch on this index (HOST out array of 16 uint64):
 * [0] search nodes expanded, [1] Occ lookups (rank queries), [2] 32-byte index sectors the rank queries read (1 per unit for blocks, 2 for lines),
 * [3] raw hits, [4] D-kernel lookups, [5] pool high-water mark, [6] search-kernel ns (CUDA events
 * on the caller's stream around the persistent search kernel), [7] geometry used:
 * ctas_per_sm << 32 | warps_per_cta << 16 | index layout << 15 | pool entries per warp, [8] warp-level branch steps,
 * [9] nodes expanded in branch steps, [10] warp-level chain iterations, [11] nodes expanded in
 * chain iterations, [12] branch states popped and put back because their children did not fit,
 * [13] 32-entry blocks of branch states spilled from the on-chip rings to the workspace,
 * [14] deepest per-warp spill stack seen (blocks), [15] bc_align_batch: blocks of 32 pending states that moved
 * from a busy warp to an idle one; bc_align_batch_best: largest per-read budget searched + 1. */
int bc_last_stats(const bc_index *ix, uint64_t *out16);

/* Tuning knobs of the persistent search kernel (0 = default: 4 CTAs per SM of 7 warps): CTAs per SM (<= 8),
 * warps per CTA (<= 8; 8 selects the kernel flavour compiled for 256 threads and 3 resident CTAs per SM). */
int bc_set_geometry(bc_index *ix, uint32_t ctas_per_sm, uint32_t warps_per_cta);

/* More tuning (0 = default): spill_blocks = per-warp spill area of the branch rings in blocks of 32
 * states (default 128; bc_align_batch returns BC_E_NOMEM when a warp's area runs full -- raise it, ask
 * bc_align_workspace_bytes again and repeat the call); pool_kb = shared memory per SM given to the
 * state pools, 16..220 KB (default: 208 KB for an index up to 64 MB, 176 KB beyond); ld_policy = cache
 * policy of the index loads: 1 = default policies, 2 = no L1 allocation + 64-byte L2 prefetch size (the library
 * default); ld_policy + 256 switches the exchange of pending states between warps off (A/B measurements).
 * spill_blocks affects the workspace size: set it before bc_align_workspace_bytes. */
int bc_set_tuning(bc_index *ix, uint32_t spill_blocks, uint32_t pool_kb, uint32_t ld_policy);

/* Device layout of indexes uploaded from now on (process-wide; 0 = by size, the default: 32-byte blocks of 64
 * symbols while the index fits 64 MB, 128-byte lines of 384 symbols beyond -- on B200 a missing 32-byte sector
 * costs a whole 128-byte line of DRAM traffic, so an index that lives in HBM makes the line its unit; 1 = blocks,
 * 2 = lines).  Read by bc_index_device_bytes and bc_index_upload.  Results do not depend on it. */
int bc_set_index_layout(int choice);

/* Host-side index construction for synthetic genomes (untimed helper): suffix sort
 * of T$ and reverse(T)$ -> transport arrays.  text: HOST, n codes 0..3.  The arrays are allocated
 * by the library and released with bc_index_host_free. */
int bc_index_build_host(const uint8_t *text, uint64_t n, uint32_t occ_interval, uint32_t sa_interval,
                        int n_threads, bc_index_host **out);
int bc_index_host_free(bc_index_host *h);

/* The same construction on the GPU: suffix arrays of T$ and reverse(T)$ by prefix
 * doubling with library radix sorts, then BWT, Occ checkpoints and SA sample in kernels.  Returns
 * transport arrays bit-identical to bc_index_build_host's (released with bc_index_host_free).
 * text: HOST, n codes 0..3; d_scratch: DEVICE, 256-byte aligned, >= bc_index_build_gpu_bytes
 * (about 34 bytes per base). */
int bc_index_build_gpu_bytes(uint64_t n, uint32_t occ_interval, uint32_t sa_interval, size_t *bytes);
int bc_index_build_gpu(const uint8_t *text, uint64_t n, uint32_t occ_interval, uint32_t sa_interval, void *d_scratch,
                       size_t scratch_bytes, void *cuda_stream, bc_index_host **out);

/* Exclusive scan of n uint32 counts into n+1 uint64 offsets (d_out[0] = 0, d_out[n] = total): the scan of step
 * A6 (per-query hit counts -> CSR offsets) on its own.  d_in, d_out, d_scratch: DEVICE; d_scratch
 * 8-byte aligned, >= bc_exclusive_scan_scratch_bytes(n) (BC_E_NOMEM otherwise).  Enqueues three kernels on the
 * stream and returns without synchronising. */
size_t bc_exclusive_scan_scratch_bytes(uint64_t n);
int bc_exclusive_scan_u32(const uint32_t *d_in, uint64_t n, void *d_scratch, size_t scratch_bytes, uint64_t *d_out,
                          void *cuda_stream);

/* The same scan for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): NO scratch argument -- the per-tile sums live in a static __device__ array inside the library
 * (262,160 bytes, held by every GPU that loads the library until the process exits), and the call performs no
 * cudaMalloc / cudaFree / allocating library call.  Limit: n <= bc_scan_static_max_n() = 67,108,864; a larger n
 * returns BC_E_UNSUPPORTED (use bc_exclusive_scan_u32 with scratch of your own).  The array's device address is
 * looked up once per device on first use (or by bc_scan_static_setup(), to be called once per device, with that
 * device current, before a stream capture starts).  All calls on a device SHARE the array and it keeps the last
 * call's contents; nothing in it needs clearing (every word read is written earlier in the same call), but calls
 * that overlap on the GPU -- two streams, two threads -- race: serialise them.  Enqueues on the stream and returns
 * without synchronising; output identical to bc_exclusive_scan_u32's. */
uint64_t bc_scan_static_max_n(void);
int bc_scan_static_setup(void);
int bc_exclusive_scan_u32_static(const uint32_t *d_in, uint64_t n, uint64_t *d_out, void *cuda_stream);

/* Measured denominator of the metric "Occ lookups/s vs the random-sector roofline":
 * every thread issues independent uniformly random 32-byte-aligned 256-bit loads (the access one
 * rank query makes) over d_table; timed with CUDA events on the stream.  d_table: DEVICE, 32-byte
 * aligned, table_bytes >= 64 (much larger than L2 => HBM rate; L2-sized => on-chip rate);
 * d_sink: DEVICE, >= 4 bytes; sectors_per_second: HOST out.  Not part of the hot path. */
int bc_measure_random_sectors(const void *d_table, size_t table_bytes, uint32_t loads_per_thread, void *d_sink,
                              void *cuda_stream, double *sectors_per_second);
/* The same with the cache policy of the load chosen: 0 = default (on B200 every L2 miss then fetches the whole
 * 128-byte line), 1 = the search kernel's default (no L1 allocation, 64-byte L2 prefetch size: 64 bytes per miss). */
int bc_measure_random_sectors2(const void *d_table, size_t table_bytes, uint32_t loads_per_thread, int ld_policy,
                               void *d_sink, void *cuda_stream, double *sectors_per_second);

const char *bc_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* BARRACUDA_B200_H */
