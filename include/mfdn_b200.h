/* mfdn_b200.h -- C ABI of libmfdn_b200.so
 *
 * Coupled-JT -> M-scheme transformation of 2- and 3-body interaction matrix elements
 * (the hot path arXiv:1412.5989 moved to the GPU inside MFDn's matrix construction),
 * B200 / sm_100a only.  No torch types, plain pointers and sizes.  Every function returns
 * MFDN_OK or a negative mfdn_status and never throws.  "PAPER.md:n" = line n of the paper
 * text; "DESIGN.md Qn" = the reading taken where the paper is silent.
 *
 * Call order:  mfdn_orbitals_init -> mfdn_cg_build -> mfdn_coupled_upload_2b / _3b ->
 *              mfdn_mscheme_2b / _3b (any number of times, any stream) -> mfdn_destroy.
 * Out-of-order calls return MFDN_ERR_STATE.
 *
 * Conventions: all indices 0-based.  Orbital o = (n, l, 2j), e = 2n+l.
 * SPS s = (orbital, 2m, 2tz), table-driven.  A request is the SPS indices of the bra then of the
 * ket ("a 3-body element request takes the form of a set of six SPS indices").
 * Canonical particle order inside a bra/ket = ascending (orbital, SPS); a request in any other
 * order is answered with the permutation sign applied.
 */
#ifndef MFDN_B200_H
#define MFDN_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mfdn_ctx mfdn_ctx; /* opaque; owns every device table */

typedef enum {
    MFDN_OK = 0,
    MFDN_ERR_ARG = -1,   /* null pointer, negative size, quantum number out of supported range */
    MFDN_ERR_STATE = -2, /* call order violated */
    MFDN_ERR_CUDA = -3,  /* a CUDA runtime call failed; see mfdn_last_error */
    MFDN_ERR_OOM = -4,   /* host or device allocation failed, or caller scratch too small */
    MFDN_ERR_TABLE = -5  /* coupled table violates its structural rules */
} mfdn_status;

/* flags of mfdn_mscheme_2b/3b */
enum {
    MFDN_PRESORTED = 1,   /* requests are already ordered by the library's sort key: NON-DECREASING mfdn_group_keys value
                             (2-body: orbital-tuple group; 3-body: group, then M; requests failing S1-S6, key
                             0xFFFFFFFF, last).  Where the library takes the group-sort path (large 3-body batches, or with
                             MFDN_FORCE_SORT) it skips the partition passes of steps H2 and H6; 3-body still histograms
                             the keys to cut the stream into one-group work items.  Input that is not so ordered gives
                             undefined VALUES on that path (never a fault); the mask stays correct */
    MFDN_FORCE_NAIVE = 2, /* one thread per request in request order, no sort, no staging: the paper's own
                             kernel design; kept as on-device reference */
    MFDN_FORCE_DENSE = 4, /* 3-body: every group whose blocks fit takes the dense-block path (step H5'): per (group, M,
                             isospin pattern) the whole block C_bra * V * C_ket^T of m-scheme elements (PAPER.md:55
                             A' = D^T A D, Fig. 1) is formed with fp64 tensor-core products (mma.sync m8n8k4) and the
                             requested entries are picked from it; the other groups take the default path.  Values
                             agree with the default path to rounding (another summation order), the mask bit for bit.
                             MFDN_ERR_ARG for 2-body calls and together with MFDN_FORCE_NAIVE */
    MFDN_ONE_PASS_SORT = 8, /* steps H2 / H6 by the one-pass scatter and gather instead of the two-pass partition through
                             shared memory.  The library takes this path by itself for tables with more than 2048 x 4096
                             sort buckets (2-body: orbital-tuple pairs; 3-body: (pair, M) combinations); the flag forces
                             it for any table (test hook and the measured baseline of DESIGN.md).  Same values bit for bit */
    MFDN_REQ_U16 = 16,     /* compact requests: d_req / h_req point to uint16 SPS indices, [n][4] or [n][6] (8 / 12 bytes per request
                             instead of 16 / 24: half the host-to-device bytes of mfdn_mscheme_host, whose time is the PCIe
                             copy).  Needs n_sps <= 65536 (else MFDN_ERR_ARG); 4-byte aligned; same results bit for bit */
    MFDN_FORCE_SORT = 32   /* take the group-sort path with the two-pass partition whatever the batch size.  Without a flag
                             that names a path the library chooses by n (all paths give the same values bit for bit):
                             2-body batches and 3-body batches of up to 2^20 requests (the ~20 000-request chunks of
                             PAPER.md:93) are evaluated thread-per-request on the library's tables, larger 3-body batches
                             by the group sort, one-pass below 2^23 requests and two-pass above */
};

/* A0. Single-particle basis (quantum numbers flattened into one linear SPS index).
 * HOST arrays, borrowed for the duration of the call.  n,l,twoj: [n_orb]; sps_*: [n_sps];
 * sps_twom odd with |2m| <= 2j, sps_twotz = +1 or -1.  Limits: n_orb <= 1023, 2j <= 21.
 * Creates the context on CUDA device `device`. */
int mfdn_orbitals_init(mfdn_ctx** out, int device, int32_t n_orb, const int32_t* n, const int32_t* l,
                       const int32_t* twoj, int32_t n_sps, const int32_t* sps_orb, const int32_t* sps_twom,
                       const int32_t* sps_twotz);

/* Options, set between mfdn_orbitals_init and the upload they concern (MFDN_ERR_STATE afterwards).
 * MFDN_OPT_SLAB_FP32 (value != 0): footprint variant of the 3-body tables (the memory
 *   footprint is the reason for coupled storage, the paper is silent on precision): the isospin-combined slabs -- the
 *   largest resident array, 4/5 of the 3-body table memory -- are STORED in fp32, every sum is still accumulated in fp64.
 *   Halves that array and the shared-memory traffic of the transform.  Values then carry the rounding of the stored
 *   numbers: |delta| <= 2^-24 * 5 max|V| per coupled cell summed, i.e. about 1e-6 max|V| instead of 1e-12 max|V|; the mask
 *   is unchanged.  MFDN_FORCE_NAIVE keeps reading the fp64 planes. */
enum { MFDN_OPT_SLAB_FP32 = 1 };
int mfdn_option(mfdn_ctx*, int option, int64_t value);

/* A1. Device-resident fp64 Clebsch-Gordan tables ("D is developed from a series of angular momentum and
 * isospin coupling coefficients"; Q1/Q2/Q10), built by one kernel from Racah's
 * formula with a double-double log-factorial table.  Asynchronous on `stream` (cudaStream_t). */
int mfdn_cg_build(mfdn_ctx*, void* stream);

/* Test hook: copy a CG table to HOST memory (synchronises).  stage 1 = <j1 m1 j2 m2|J M> for half-integer
 * j1,j2 <= jmax; stage 2 = <J12 M12 j m|J M> for integer J12 <= 2*jmax and half-integer j <= jmax.
 * Layout: blocks in ascending (first, second) angular momentum order; stage-1 block (2j1,2j2) holds
 * [iJ][i1][i2] (i2 fastest), i = (2m+2j)/2, iJ = (2J - |2j1-2j2|)/2, value <j1 m1 j2 m2|J m1+m2>
 * (0 where |m1+m2| > J); stage-2 block (J12, 2j) likewise with j1 = J12.
 * *n receives the entry count; if host_out is NULL or cap < *n nothing is copied. */
int mfdn_cg_download(mfdn_ctx*, int stage, double* host_out, int64_t cap, int64_t* n);

/* A2. Coupled-JT tables, channel-major (only potentially-nonzero elements, one block per
 * orbital combination).  chan_* have length n_chan; state_* have length sum(chan_dim), listed channel by
 * channel; channel c is a row-major chan_dim[c] x chan_dim[c] fp64 square at values + chan_off[c].
 * Index arrays are HOST; `values` is HOST or DEVICE (values_on_device != 0).  The library copies and
 * re-tiles (group-major, in the order the kernel's nested loops read them) and, for 3-body tables,
 * builds the per-tuple coefficient tables <ja ma jb mb|J12 M12><J12 M12 jc mc|J M>; the caller keeps ownership.  Structural rules (else MFDN_ERR_TABLE): orbitals in range and a <= b (<= c); triangle rules;
 * channel parity = parity of the state's orbitals; a == b only with J+T (2-body) resp. J12+T12 (3-body) odd;
 * 3-body: e_a+e_b+e_c <= e3max, 2T in {1,3}, T12 in {0,1}; no duplicate channel or state; (2ja+1)(2jb+1)(2jc+1) <= 4096
 * for every listed orbital triple (12-bit m-state index of the packed request record).
 * 2-body: chan_J, chan_T are J and T; 3-body: chan_twoJ, chan_twoT are 2J and 2T.  chan_par: 0 even, 1 odd.
 * Synchronises `stream` before returning. */
int mfdn_coupled_upload_2b(mfdn_ctx*, int32_t n_chan, const int32_t* chan_J, const int32_t* chan_T,
                           const int32_t* chan_par, const int32_t* chan_dim, const int64_t* chan_off,
                           const int32_t* state_a, const int32_t* state_b, const double* values,
                           int values_on_device, void* stream);
int mfdn_coupled_upload_3b(mfdn_ctx*, int32_t e3max, int32_t n_chan, const int32_t* chan_twoJ,
                           const int32_t* chan_twoT, const int32_t* chan_par, const int32_t* chan_dim,
                           const int64_t* chan_off, const int32_t* state_a, const int32_t* state_b,
                           const int32_t* state_c, const int32_t* state_J12, const int32_t* state_T12,
                           const double* values, int values_on_device, void* stream);

/* H1-H6. The transformation (formulas in DESIGN.md "What is computed").
 * d_req : DEVICE int32 [n][4] = (bra0,bra1,ket0,ket1)  /  [n][6] = (bra0..2, ket0..2); 16-byte aligned.
 * d_out : DEVICE double [n]; d_mask: DEVICE uint8 [n] or NULL.  Caller-owned, results in REQUEST order.
 *         mask[i] = 1 iff the request passes the integer selection rules S1-S7; where
 *         mask[i] = 0 the value is exactly +0.0.
 * d_work/work_bytes: caller-provided DEVICE scratch, 256-byte aligned.  Call with d_work == NULL to get
 *         the size needed for n requests WITH THESE FLAGS in *work_bytes (nothing is launched; the size depends on both).  The call itself never
 *         allocates and never synchronises: it is asynchronous on `stream`.
 * Per-request problems never fail the call: an out-of-range SPS index gives value 0, mask 0 and is
 * counted (mfdn_bad_request_count).  Concurrent calls are allowed -- from one host thread or from several -- provided
 * each call in flight has its own stream and its own scratch (one stream per host thread); the tables
 * are read-only and the context's bookkeeping is locked.  The call makes the context's device the calling thread's
 * current device. */
int mfdn_mscheme_2b(mfdn_ctx*, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                    size_t* work_bytes, uint32_t flags, void* stream);
int mfdn_mscheme_3b(mfdn_ctx*, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                    size_t* work_bytes, uint32_t flags, void* stream);

/* The step that follows the transformation in MFDn, fused into the call.  PAPER.md:93: every
 * buffered request carries "which many-body element the request pertains to" and "a specific phase"; the host
 * "iterates through the returned three-body elements in the chunk, multiplies them by the stored phases, and adds them to
 * the array of many-body elements at the stored locations".  Here the results are not returned:
 *     d_H[d_loc[i]] += d_phase[i] * v_i      for every request i with 0 <= d_loc[i] < h_len,
 * v_i being what mfdn_mscheme_2b/3b would have written to d_out[i].
 * d_loc  : DEVICE int64 [n], index into d_H; an entry outside [0, h_len) is skipped (its mask is still written).
 * d_phase: DEVICE double [n] or NULL (= +1 everywhere).   d_H: DEVICE double [h_len], caller-owned and caller-initialised;
 *          it is updated with fp64 atomic adds, so concurrent calls may target the same array; the order of the additions
 *          to one element is not fixed (results agree to rounding from run to run, not bit for bit).
 * Everything else (d_req, d_mask, scratch query with d_work == NULL, flags, stream, error behaviour) as for mfdn_mscheme_2b/3b;
 * the scratch size differs from theirs. */
int mfdn_mscheme_accumulate_2b(mfdn_ctx*, int64_t n, const int32_t* d_req, const int64_t* d_loc, const double* d_phase,
                               double* d_H, int64_t h_len, uint8_t* d_mask, void* d_work, size_t* work_bytes, uint32_t flags,
                               void* stream);
int mfdn_mscheme_accumulate_3b(mfdn_ctx*, int64_t n, const int32_t* d_req, const int64_t* d_loc, const double* d_phase,
                               double* d_H, int64_t h_len, uint8_t* d_mask, void* d_work, size_t* work_bytes, uint32_t flags,
                               void* stream);

/* Dense block mode: whole m-scheme blocks without a request list -- the block view A' = D^T A D of
 * PAPER.md:55 (Fig. 1 at :69), for use "at a higher level in the matrix construction stage"; trades the
 * memory blow-up of PAPER.md:53 for bandwidth.  A block belongs to a pair of 3-body orbital tuples, bra (a <= b <= c) and ket
 * (d <= e <= f): `orbitals` = {a, b, c, d, e, f}.  Its entries, in this order:
 *   for mi = 0 .. mm          common M ascending: mm = min(ja+jb+jc, jd+je+jf) (2j units), 2M = 2 mi - mm
 *     for bin = 0 .. 19       isospin patterns: the pairs (pb, pk), pb = ta<<2 | tb<<1 | tc of the bra (bit = 1 for 2tz = +1),
 *                             pk likewise for the ket, with equally many set bits, in ascending (pb, pk) order
 *       an nb x nk matrix, row-major: rows = the bra m-states (ma, mb, mc) of that M in ascending (ia, ib) order
 *                             (i = (2m + 2j) / 2), columns = the ket m-states likewise
 * entry = < a ma ta, b mb tb, c mc tc | V | d .., e .., f .. >, i.e. what mfdn_mscheme_3b returns for that request, if bra
 * and ket are ordered Slater determinants (all six SPS exist; particles of one orbital in ascending SPS index order);
 * otherwise +0.0 (the value is that of the ordered partner times the permutation sign).  Entries forbidden by a selection
 * rule are +0.0 as well.  The block is empty (length 0, nothing written) if a tuple is not listed in the uploaded table,
 * the parities differ or there is no common J.
 * mfdn_mscheme_block_len_3b: HOST call, *n_values = number of doubles of the block.
 * mfdn_mscheme_blocks_3b: n_groups blocks in one launch; h_orbitals: HOST int32 [n_groups][6]; h_off: HOST int64
 *   [n_groups], offset (in doubles) of every block in d_out (DEVICE, caller-owned, large enough); d_work/work_bytes:
 *   DEVICE scratch, queried with d_work == NULL; asynchronous on `stream` (the host arrays may be reused on return).
 *   Formed with fp64 tensor-core products (mma.sync m8n8k4): values agree with mfdn_mscheme_3b to rounding.
 *   MFDN_ERR_ARG for orbitals out of range or not ascending and for a group with more than 64 ket rows (J, J12'). */
int mfdn_mscheme_block_len_3b(mfdn_ctx*, const int32_t* orbitals, int64_t* n_values);
int mfdn_mscheme_blocks_3b(mfdn_ctx*, int64_t n_groups, const int32_t* h_orbitals, const int64_t* h_off, double* d_out,
                           void* d_work, size_t* work_bytes, void* stream);

/* The paper's wrapper ("transfer a chunk of 3-body element requests to the GPU, invoke the kernel,
 * and transfer the results back"), for HOST request/result buffers (pinned memory recommended).  The n requests
 * are cut into chunks of `chunk` (0 = library default) and H2D copy / transform / D2H copy of successive chunks
 * overlap on four internal streams.  body = 2 or 3; h_mask may be NULL; flags as above (MFDN_PRESORTED then means
 * the whole host array is group-ordered).  d_work/work_bytes: DEVICE scratch, queried with d_work == NULL.
 * BLOCKING: returns after the last result byte has landed in h_out (also on failure: no copy is left in flight on the
 * caller's buffers).  Uses four streams owned by the context: one mfdn_mscheme_host call at a time per context. */
int mfdn_mscheme_host(mfdn_ctx*, int body, int64_t n, const int32_t* h_req, double* h_out, uint8_t* h_mask,
                      void* d_work, size_t* work_bytes, uint32_t flags, int64_t chunk);

/* The allocation-free call, for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): mfdn_mscheme_2b/3b (the same steps H1-H6, the same kernels, the
 * same values bit for bit) with the scratch the group-sort path needs taken from an array that is PART OF THE LIBRARY
 * instead of from the caller: MFDN_STATIC_SCRATCH_BYTES of device memory, which every GPU that loads the library holds until
 * the process exits.  body = 2 or 3; d_req, d_out, d_mask (may be NULL), flags and stream as for mfdn_mscheme_2b/3b;
 * asynchronous on `stream`.  It calls no cudaMalloc, cudaFree or other allocating routine.
 *  - The first call on a device looks up the array's device address once (cudaGetSymbolAddress, with that device
 *    current); a call with n = 0 does just that and is the set-up call to make before a capture or a timed loop.
 *  - A batch that needs more scratch than the array holds is rejected with MFDN_ERR_OOM (mfdn_last_error names both
 *    sizes): the need is what mfdn_mscheme_2b/3b report for the same (n, flags) with d_work == NULL, about 45 bytes per
 *    3-body request on the group-sort path plus 4 bytes per sort bucket of the table (config 3: 6.4 MB + n * 45 B, i.e. up
 *    to ~5 * 10^5 requests per call; config 4, 7.7 M buckets = 30.7 MB: ~6 * 10^4; the paper's request buffers hold
 *    ~20 000).  2-body batches and 3-body
 *    batches of up to 2^20 requests are evaluated thread per request unless a flag names the sort path, and need none.
 *  - MFDN_ERR_STATE while mfdn_profile is on (profiling creates events).
 *  - EVERY call in the process, from any context on the same device, uses the SAME array, and the array keeps the
 *    last call's contents: the call clears what must start at zero (histogram, work-item counters) itself, on `stream`;
 *    two calls that overlap on the GPU (different streams, or different host threads) race on it and give undefined
 *    values.  Calls on one stream are ordered and safe. */
#define MFDN_STATIC_SCRATCH_BYTES (32u << 20)
int mfdn_mscheme_static(mfdn_ctx*, int body, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, uint32_t flags,
                        void* stream);

/* Measurement hooks.  mfdn_profile(ctx, 1) makes every later mfdn_mscheme_2b/3b call record CUDA events on the
 * call's stream around (1) its group-sort kernels (H1-H2: keys, scans, partition passes, work-item list), (2) its transform
 * kernel (H3-H6) and (3) the gather of the results back into request order (sort path only; 0 for MFDN_PRESORTED
 * and MFDN_FORCE_NAIVE).  mfdn_profile_read synchronises those events, returns the accumulated milliseconds of the
 * three parts and the call count since the last read, and resets them.  mfdn_fp64_peak runs a register-resident
 * DFMA micro-benchmark on all SMs (the fp64 roofline denominator; MEASURED_PEAKS.json has no fp64 entry) and
 * returns TFLOP/s (2 flops per FMA); synchronises. */
/* mfdn_multi_client (SURVEY.md 8(f) NEXT-3; PAPER.md:93 request buffers of ~20 000 entries, :103 "each OpenMP thread is given
 * its own stream"): n_threads host threads (<= 64) created by the call, each with its own stream and its own scratch, push
 * the n DEVICE-resident requests through the context in chunks of `chunk` (thread t takes chunks t, t + n_threads, ...);
 * d_out / d_mask receive the results as from one big call.  *seconds = wall clock of the whole job.  BLOCKING; allocates
 * and frees its streams and scratch. */
int mfdn_multi_client(mfdn_ctx*, int body, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, int64_t chunk,
                      int n_threads, uint32_t flags, double* seconds);
int mfdn_profile(mfdn_ctx*, int enable);
int mfdn_profile_read(mfdn_ctx*, double* ms_sort, double* ms_transform, double* ms_unpermute, int64_t* calls);
int mfdn_fp64_peak(mfdn_ctx*, double* tflops);

/* Number of requests with an out-of-range SPS index seen so far (synchronises `stream`). */
int64_t mfdn_bad_request_count(mfdn_ctx*, void* stream);

/* Sizes of what was uploaded, for reports: which = 0 tuples (2b), 1 tuples (3b), 2 slab bytes (2b),
 * 3 slab bytes (3b), 4 CG entries stage 1, 5 CG entries stage 2, 6 kernels launched so far by mscheme_*, 7 bytes of the
 * 3-body coefficient tables, 8 bytes of the 3-body isospin-combined slabs, 9 number of 3-body (group, M) sort buckets. */
int64_t mfdn_info(mfdn_ctx*, int which);

/* Sort key of every request, for producing MFDN_PRESORTED input (sort ascending by it): 2-body d_key[i] = bra_tuple *
 * n_tuples + ket_tuple; 3-body the (group, M) bucket = first bucket of the group bra_tuple * n_tuples + ket_tuple + index
 * of the request's M in the group's common M range (requests of one group are contiguous, ordered by M: the
 * coefficient tables are M-major, so neighbouring requests read neighbouring entries).  0xFFFFFFFF for requests that
 * fail S1-S6.  body = 2 or 3; d_req holds int32 indices (no MFDN_REQ_U16 form).  Asynchronous on `stream`. */
int mfdn_group_keys(mfdn_ctx*, int body, int64_t n, const int32_t* d_req, uint32_t* d_key, void* stream);

/* Message of the context's most recent failure; the pointer stays valid until the calling thread's next call of this function. */
const char* mfdn_last_error(mfdn_ctx*);
void mfdn_destroy(mfdn_ctx*);

#ifdef __cplusplus
}
#endif
#endif /* MFDN_B200_H */
