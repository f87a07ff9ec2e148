/*
 * ccl.h -- C ABI of libccl.so: bond-list connected-component labeling for sm_100a (NVIDIA B200).
 *
 * The operation is the hot path of Y. Komura, "A generalized GPU-based connected component labeling
 * algorithm" (arXiv 1603.08357; PAPER.md), section 3: four steps -- (i) initialization, (ii) analysis,
 * (iii) label reduction with atomicMin (Algorithm 1), (iv) analysis --
 * with the nearest-neighbour list of PAPER.md:111 replaced by a bond list plus per-bond occupancy
 * (BASELINE.json north_star).  The result is the canonical labeling of PAPER.md:115:
 *
 *        labels[i] = smallest site index in the connected component of site i.
 *
 * Conventions for every entry point
 *   - All array pointers are DEVICE pointers owned by the caller unless the name says `host_`.  The library
 *     never frees caller memory.  Scratch a call needs comes from the library's own stream-ordered memory pool
 *     (one cudaMemPool_t per device, cudaMallocFromPoolAsync) and is returned to that pool, in stream order, before
 *     the call returns.  The pool KEEPS what it has reserved for the next call (so that a sweep of calls does not
 *     pay the driver for memory each time) until ccl_trim_scratch() hands it back; ccl_scratch_bytes() reports it.
 *     What a call draws: ccl_label / ccl_label_bits nothing, unless n_sites * 4 >= 96 MiB and n_bonds >= 2^20 (the
 *     region-bucketed form): then 10 * n_bonds bytes of pair chunks plus a table (about 1.5 GB for 2^27 bonds; twice,
 *     four, at most eight times that on a bond list on which an earlier call ran the pool dry) -- except that a call
 *     on a bond list for which the remembered probe answer is "direct" draws nothing, and that a call whose workspace
 *     cannot be allocated does not fail: it runs the direct kernels, which need none;
 *     the host-buffer entry points also their device copies of src, dst, masks and labels.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the default stream).  All work is enqueued on it; no
 *     entry point synchronises with the host unless stated.  Results are valid once the stream has drained.
 *   - Return value: CCL_OK (0) or a ccl_status.  No exception crosses the ABI.  ccl_last_error() returns a
 *     thread-local, NUL-terminated description of the last failure on the calling thread.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns CCL_CUDA_ERROR.
 */
#ifndef CCL_H_
#define CCL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ccl_status {
    CCL_OK = 0,
    CCL_INVALID_ARG = 1,          /* negative count, count > 2^31-1 sites, NULL where data is required */
    CCL_CUDA_ERROR = 2,           /* a CUDA runtime call or launch failed; see ccl_last_error()         */
    CCL_UNSUPPORTED = 3,          /* argument combination the library does not implement               */
    CCL_WORKSPACE_TOO_SMALL = 4   /* caller-provided workspace is smaller than the size query reported  */
} ccl_status;

/* Result of ccl_cluster_stats (reading R8).  Lives in device memory; 32 bytes. */
typedef struct ccl_stats {
    int64_t  n_clusters;      /* #{ i : labels[i] == i }                                             */
    int64_t  largest;         /* size of the largest cluster                                          */
    int64_t  largest_label;   /* its label; ties broken towards the smallest label                    */
    uint64_t sum_s2;          /* sum over clusters of size^2 (<= N^2 < 2^63 for N <= 2^31)             */
} ccl_stats;

/* ---- the hot path: steps (i)-(iv), PAPER.md:113 ------------------------------------------------------
 *
 * ccl_label: bonds b = 0..n_bonds-1 join sites src[b] and dst[b] (two separate int32 arrays); bond b is
 * occupied iff occupied[b] != 0 (one uint8 per bond); occupied == NULL means every bond is occupied.
 * labels[n_sites] (int32) is write-only on entry -- no initial content is required -- and holds the canonical
 * labels on completion; it must be 16-byte aligned (else CCL_INVALID_ARG; every cudaMalloc / torch allocation is).
 * src, dst, occupied are read-only and may have any alignment (16-byte aligned src/dst take the vectorised path).  0 <= src[b], dst[b] < n_sites is a caller
 * precondition that is NOT checked here (use ccl_validate_bonds).  Self-loops and repeated bonds are legal.
 * n_bonds == 0 gives labels[i] = i.  n_sites == 0 is a no-op.  The result does not depend on bond order.
 * Errors: n_sites < 0, n_sites > 2^31-1, n_bonds < 0, NULL src/dst/labels with a non-zero count, or misaligned
 * labels -> CCL_INVALID_ARG.
 * The library remembers, per host thread, what its device-side probe said about the last few bond lists (keyed by
 * the src/dst pointers and the counts) and skips the probe on later calls; this changes speed only, never results.
 */
int ccl_label(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
              const uint8_t* occupied, int32_t* labels, void* stream);

/* Same with a packed mask: bond b is bit (b & 31) of uint32 word (b >> 5); ceil(n_bonds/32) words (4-byte aligned),
 * bits past n_bonds are ignored. */
int ccl_label_bits(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                   const uint32_t* occupied_bits, int32_t* labels, void* stream);

/* The paper's own interface: a nearest-neighbour list instead of a bond list.  nn_list is a dense
 * z_max x n_sites int32 array, structure of arrays: the k-th neighbour of site i is nn_list[k * n_sites + i]; negative
 * entries are padding.  Every entry is a connection of the network to be labeled; a bond may be listed at both of its
 * ends (the paper's form) or at either one.
 * The four steps run in the paper's form: (i) label[i] = smallest lower-numbered neighbour, else i; (ii) analysis;
 * (iii) Algorithm 1 over every listed entry (site i, neighbour j != i), whichever of the two is lower -- so a bond listed
 * at one end only is still joined; (iv) analysis.  Same result as ccl_label on the
 * corresponding bond list.  0 <= z_max <= 1024; neighbours >= n_sites are a caller error (not checked). */
int ccl_label_nn(int64_t n_sites, int32_t z_max, const int32_t* nn_list, int32_t* labels, void* stream);

/* Debug validator: *out_bad (device int64) = number of bonds with an endpoint outside [0, n_sites). */
int ccl_validate_bonds(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                       int64_t* out_bad, void* stream);

/* ---- seeded workload generators (outside the timed metric) -----------------
 *
 * Periodic L x L lattices, 3*L*L bonds each (the paper names the lattices only; geometry and
 * numbering are this project's, reading R9):
 *   triangular: site s = y*L + x; bond 3s+k joins s to (x+1,y), (x,y+1), (x+1,y+1) mod L for k = 0,1,2.
 *   honeycomb : cell c = y*L + x holds sites A = 2c, B = 2c+1; bond 3c+0 = A(c)-B(c), 3c+1 = B(c)-A(x+1,y),
 *               3c+2 = B(c)-A(x,y+1) mod L; src is the first-named site.
 * L >= 1 and 2*L*L <= 2^31-1.
 */
int ccl_gen_triangular(int32_t L, int32_t* src, int32_t* dst, void* stream);
int ccl_gen_honeycomb(int32_t L, int32_t* src, int32_t* dst, void* stream);

/* Cayley tree with coordination number 3 and g generations -- the paper's own "Bethe lattice" workload
 * (PAPER.md:189-193): N = 3*2^g - 2 sites, N - 1 bonds; site 0 has children 1, 2, 3 and site i >= 1 has children
 * 2i+2, 2i+3 ("standard position" numbering, R11); bond k joins site k+1 (dst) to its parent (src).
 * perm_or_null: device int32[N] permutation giving the "random" numbering (site i is called perm[i]); NULL = standard.
 * 1 <= g <= 28. */
int ccl_gen_cayley3(int32_t g, const int32_t* perm_or_null, int32_t* src, int32_t* dst, void* stream);

/* Simple random z-regular graph on n_sites sites by the configuration model ("Bethe substitute" of
 * BASELINE.json configs 4-5; the paper's own Bethe workload is the Cayley tree):
 * n_sites*z/2 bonds in uniformly random order; stub keys from Philox4x32-10, stable sort, defects (self-loops,
 * repeated pairs) repaired by seeded endpoint swaps.  Call with workspace == NULL to obtain the required size in
 * *workspace_bytes (host pointer); then call again with a device workspace of at least that size.
 * n_sites*z must be even, 1 <= z <= 16, n_sites*z <= 2^31-1. */
int ccl_gen_regular(int64_t n_sites, int32_t z, uint64_t seed, int32_t* src, int32_t* dst,
                    void* workspace, size_t* workspace_bytes, void* stream);

/* Bernoulli(p) occupancy: T = floor(p*2^32) computed on the host in double; bond b is occupied iff word (b & 3)
 * of Philox4x32-10(counter = (b>>2 lo, b>>2 hi, realization, 0), key = (seed lo, seed hi)) < T; p >= 1 occupies
 * everything.  Writes whichever of the two outputs is non-NULL: a uint8 0/1 mask [n_bonds] and/or packed bits
 * [ceil(n_bonds/32) words, unused high bits zero].  The same seed at two values of p gives nested sets. */
int ccl_gen_occupancy(int64_t n_bonds, double p, uint64_t seed, uint32_t realization,
                      uint8_t* mask_or_null, uint32_t* bits_or_null, void* stream);

/* ---- cluster statistics from canonical labels (outside the timed metric) -----------------------------
 *
 * size_scratch: device int32[n_sites], overwritten (cluster sizes indexed by label).  out: device ccl_stats.
 * hist_dense (optional): device int64[n_dense+1]; hist_dense[s] = number of clusters of size exactly s,
 * 1 <= s <= n_dense; entry 0 is set to 0.  hist_log2 (optional): device int64[32]; hist_log2[k] = number of
 * clusters with 2^k <= size < 2^(k+1).  labels must be canonical (output of ccl_label*). */
int ccl_cluster_stats(int64_t n_sites, const int32_t* labels, int32_t* size_scratch, ccl_stats* out,
                      int64_t* hist_dense, int32_t n_dense, int64_t* hist_log2, void* stream);

/* ---- the same statistics without any device allocation ------------------------------------------------
 *
 * For callers that cannot allocate device memory and so cannot bring the size_scratch ccl_cluster_stats asks for:
 * a program that gave the whole GPU to its own memory arena at start-up (cudaMalloc would fail), or a loop that must
 * not issue cudaMalloc / cudaFree because both synchronise the device and stall every other stream of the process.
 * The per-label size table lives in a fixed array inside the library image instead: CCL_STATS_STATIC_MAX_SITES int32
 * counters = 16 MiB, held on every GPU that loads libccl.so from module load until the process exits.  The call
 * itself issues no cudaMalloc, cudaFree, memory-pool or other allocating call; it enqueues memsets and the kernels
 * of ccl_cluster_stats on `stream`.  labels, out, hist_dense, n_dense, hist_log2: as for ccl_cluster_stats, all
 * caller-owned device memory; same results.
 *   - n_sites > CCL_STATS_STATIC_MAX_SITES -> CCL_INVALID_ARG (checked on the host before anything is enqueued;
 *     use ccl_cluster_stats with your own scratch for larger label arrays).
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current) and caches it; make that first call during set-up, before any stream capture is begun.
 *   - Every call on a device uses the SAME array.  The call clears the n_sites counters it needs, so earlier
 *     contents never leak into a result, but two calls whose kernels overlap on the GPU (different streams, or
 *     different host threads on different streams) race on it and both results are garbage: keep calls on one
 *     device in one stream order. */
#define CCL_STATS_STATIC_MAX_SITES (1 << 22)
int ccl_cluster_stats_static(int64_t n_sites, const int32_t* labels, ccl_stats* out, int64_t* hist_dense,
                             int32_t n_dense, int64_t* hist_log2, void* stream);

/* ---- whole-call convenience with HOST buffers (the end-to-end path bench.py times as "e2e") ----------
 *
 * Copies src/dst/occupied_bits from host memory (pinned for full speed) to device scratch the call allocates and
 * frees, runs ccl_label_bits, copies labels back to host_labels and synchronises the stream before returning. */
int ccl_label_bits_host(int64_t n_sites, int64_t n_bonds, const int32_t* host_src, const int32_t* host_dst,
                        const uint32_t* host_occupied_bits, int32_t* host_labels, void* stream);

/* ---- wrapping on a periodic lattice (reading R7 of "spanning") ---------------
 *
 * ccl_gen_wrap_vectors: per bond of ccl_gen_triangular (family 0) / ccl_gen_honeycomb (family 1), in the same bond
 * order, how many times the bond crosses the periodic seam from src to dst along x and along y (0 or 1 here; ccl_wrap
 * accepts -1, 0, 1).  int8 [3*L*L] each.
 *
 * ccl_wrap: out[0] = 1 iff some cluster of the occupied graph holds a closed path with non-zero winding along x, out[1]
 * the same along y, out[2] = 1 iff an internal 16-bit sheet offset overflowed (result invalid; needs > 32000 seam
 * crossings on one path), out[3] = 0.  out: device int32[4].  Method: labels_open (device int32[n_sites], output)
 * receives the canonical labels of the OPEN lattice (occupied bonds with a zero wrap vector, through ccl_label_bits);
 * the occupied seam bonds then run a lock-free weighted union-find over the open clusters.  wx, wy: device int8
 * [n_bonds], 16-byte aligned.  occupied_bits as in ccl_label_bits (NULL = all occupied).  workspace: call with
 * workspace == NULL for the size in *workspace_bytes (host pointer); 256-byte aligned device memory. */
int ccl_gen_wrap_vectors(int32_t family, int32_t L, int8_t* wx, int8_t* wy, void* stream);
int ccl_wrap(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const uint32_t* occupied_bits,
             const int8_t* wx, const int8_t* wy, int32_t* labels_open, int32_t* out, void* workspace,
             size_t* workspace_bytes, void* stream);

/* ---- many realizations of one small graph in one launch ---------------------------
 *
 * The same bond list (src, dst, n_bonds) under n_batch packed occupancy masks: realization r reads the mask at
 * occupied_bits + r * mask_stride_words (bond b = bit (b & 31) of word (b >> 5); NULL = every bond occupied in every
 * realization) and writes labels[r * n_sites .. (r+1) * n_sites).  One CTA per realization runs steps (i)-(iv) of
 * PAPER.md:113 with the whole label array in shared memory, so n_sites <= 32768 (else CCL_UNSUPPORTED: call
 * ccl_label_bits per realization).  Percolation studies average many independent realizations; a single
 * call on a lattice this small is bound by launch latency.  Same result per realization as ccl_label_bits. */
int ccl_label_batch(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                    const uint32_t* occupied_bits, int64_t mask_stride_words, int32_t n_batch, int32_t* labels,
                    void* stream);

/* ---- sequential cluster numbers ("to assign the labels sequentially ...") -----------------
 *
 * labels: canonical labels (output of ccl_label*).  seq_labels[i] = number of clusters whose label is smaller than
 * labels[i], i.e. clusters numbered 0..C-1 in ascending order of their smallest site; *n_clusters (device int64,
 * optional) = C.  seq_labels may alias labels.  Call with workspace == NULL to obtain the required size in
 * *workspace_bytes (host pointer), then again with a device workspace of at least that size. */
int ccl_relabel_sequential(int64_t n_sites, const int32_t* labels, int32_t* seq_labels, int64_t* n_clusters,
                           void* workspace, size_t* workspace_bytes, void* stream);

/* An occupancy sweep over ONE bond list with host buffers (BASELINE.json configs 3 and 5 sweep p): the bond list is
 * copied to the device once, mask k is labeled while the labels of mask k-1 travel back on a second stream.
 * host_occupied_bits / host_labels: host arrays of n_masks host pointers (a NULL mask = every bond occupied; label
 * buffers of n_sites int32 each).  Synchronises before returning.  Same results as n_masks ccl_label_bits_host calls. */
int ccl_label_sweep_host(int64_t n_sites, int64_t n_bonds, const int32_t* host_src, const int32_t* host_dst,
                         int32_t n_masks, const uint32_t* const* host_occupied_bits, int32_t* const* host_labels,
                         void* stream);

/* ---- scratch memory ---------------------------------------------------------------------------------------
 *
 * ccl_trim_scratch: synchronises `stream`, then returns to the driver all memory the library's pool on the current
 * device holds beyond keep_bytes (0 = everything that is not in use).  ccl_scratch_bytes: bytes the pool has
 * reserved from the driver / bytes currently handed out to calls in flight (either pointer may be NULL; host pointers). */
int ccl_trim_scratch(size_t keep_bytes, void* stream);
int ccl_scratch_bytes(int64_t* reserved, int64_t* in_use);

/* ---- tuning --------------------------------------------------------------------------------------------
 *
 * ccl_set_option(name, value): knobs of the CALLING HOST THREAD (like ccl_last_error and ccl_launch_count; a call
 * reads them once on entry, so another thread can never change a call in flight); none of them changes the result of
 * ccl_label.  Step (iii) has two forms: the direct kernels, and a region-bucketed form for label
 * arrays too large for L2, which a device-side probe selects when the bonds are not local in the site numbering.
 *   "bucket_min_label_bytes"  label arrays of at least this many bytes are eligible for the bucketed form
 *                             (default 96 MiB; 0 makes every call eligible; negative restores the default)
 *   "region_shift"            a region is 2^value sites (default 23, allowed 4..30; raised automatically so that
 *                             there are at most 32 regions; negative restores the default)
 *   "force_mode"              -1 = the probe decides (default), 0 = always direct, 1 = always bucketed when eligible
 *   "bucket_capacity"         pairs the chunk pool of the bucketed form can hold (<= 0: 1.25 n_bonds + slack, doubled
 *                             for later calls on a bond list whenever it ran dry); if it runs dry the direct kernel
 *                             re-does the bond list behind the bucketed kernels
 *   "scatter_tiles"           1 = the bulk-copy (cp.async.bulk) scatter kernel for 16-byte aligned input (default),
 *                             0 = the register kernel for everything
 *   "probe_cache"             1 = remember the probe's answer per bond list (default), 0 = probe on every call;
 *                             setting it (either way) forgets what this thread remembers about earlier bond lists
 *   "two_pass"                direct form of step (iii): 0 = one pass over the bonds, 1 = the paper's order of work
 *                             (hook every site to its smallest lower neighbour, flatten, then Algorithm 1; two passes
 *                             over the bonds), -1 = two passes iff n_bonds >= 2.5 n_sites and n_bonds >= 2^20 (default)
 *   "flatten_window_bytes"    step (iv) behind the bucketed form gathers from one window of label[] of this many bytes
 *                             at a time (default 64 MiB, what stays resident in L2);
 *   "flatten_window_min_bytes" ... for label arrays of at least this many bytes (default 96 MiB; 0 = always; < 0 = never)
 *   "l2_persist"              1 = the k_descend and windowed k_flatten launches of the bucketed form carry a per-launch
 *                             access-policy window (persisting) over the slice of labels[] they work on.  Default 0:
 *                             measured slower on B200 (profiles/r3_l2_window.md).  SIDE EFFECT when on: the first such
 *                             call raises the device-wide limit cudaLimitPersistingL2CacheSize to the device's maximum
 *                             (79 MiB of the 126.5 MiB L2 on B200), which stays in force for the whole process
 *   "reset"                   all defaults (value ignored); also forgets the remembered bond lists
 * Unknown names -> CCL_INVALID_ARG. */
int ccl_set_option(const char* name, int64_t value);

/* ---- profiling hook ------------------------------------------------------------------------------------
 *
 * Optional cudaEvent_t handles (as void*, any of them NULL = off) that the NEXT ccl_label / ccl_label_bits calls on
 * this host thread record on their stream: after step (i) (k_init; when the bucketed kernels write the labels
 * region by region themselves there is no separate step (i) and the event falls at the start of step (iii)), after
 * step (iii) and after step (iv) (k_flatten).  Together with an event the caller records before the call they give each step's device time
 * from inside the caller's own timed region.  The handles stay in force until replaced; pass three NULLs to clear. */
int ccl_set_profile_events(void* after_init, void* after_reduce, void* after_flatten);

/* ---- diagnostics ------------------------------------------------------------------------------------- */
const char* ccl_last_error(void);      /* thread-local; never NULL                                      */
int ccl_version(void);                 /* 10000*major + 100*minor + patch                                */
/* Number of kernels this library has launched on the calling thread since load (bench.py's gpu_launches). */
int64_t ccl_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* CCL_H_ */
