/* include/lst.h -- C ABI of the B200-native line-segment-tracking (LST) hot path.
 *
 * What the library computes: the segment-building chain of arXiv:2403.13166 for one event's
 * outer-tracker hits -- mini-doublets, line segments, triplets, quintuplets, the T5-DNN score of
 * every quintuplet and the four mutually exclusive track-candidate types (Table 1,
 * PAPER.md:45-60; T5-DNN PAPER.md:62-68, :90).  The cuts the paper leaves out are frozen in
 * SPEC.md; section numbers below refer to it.  Entry-point names follow BASELINE.json north_star (1):
 * lst_create / lst_load_event / lst_run / lst_get.
 *
 * Conventions
 *  - Every function returns LST_OK (0) or a negative error; none throws, aborts or prints.
 *  - "HOST" / "DEVICE" on a pointer says where the memory lives.  The caller owns ALL memory:
 *    the library allocates nothing on the device; it carves the caller's workspace.
 *  - `cuda_stream` is a cudaStream_t passed as void* (torch.cuda.Stream().cuda_stream); 0 = default
 *    stream.  lst_load_event*, lst_run* and lst_read_* only ENQUEUE work; lst_status synchronises.
 *  - A context holds `n_slots` independent event slots that share one uploaded geometry
 *    (BASELINE.json configs[3]: "geometry and connectivity uploaded once").
 *  - Threads: a context is NOT thread-safe.  lst_run_batch keeps a cache of captured launch graphs and shares one
 *    capture side-stream per context, so all calls on one context must come from one host thread at a time (the paper's
 *    own usage: one host thread per stream -- give each thread its own context, they share nothing).
 *  - Overflow of a stage capacity is NOT an error return: the stage keeps the first `cap` objects in
 *    build order and sets its bit in the slot's status word (SPEC.md 6) -- flagged, never silent.
 */
#ifndef LST_H_
#define LST_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LST_OK 0
#define LST_EINVAL (-1)  /* null pointer, size above capacity, malformed CSR, bad slot / objtype   */
#define LST_ECUDA (-2)   /* a CUDA runtime call failed (sticky)                                   */
#define LST_ENOMEM (-3)  /* workspace smaller than lst_workspace_bytes()                          */
#define LST_ETOOBIG (-4) /* lst_sort_hits_static only: input larger than its fixed built-in scratch   */

/* status bits (lst_status) */
#define LST_ST_BAD_KEY (1u << 0)   /* a hit key >= 2*n_modules was dropped (SPEC.md 4.0)          */
#define LST_ST_OVF_MD (1u << 1)
#define LST_ST_OVF_LS (1u << 2)
#define LST_ST_OVF_T3 (1u << 3)
#define LST_ST_OVF_T5C (1u << 4)
#define LST_ST_OVF_T5 (1u << 5)
#define LST_ST_OVF_TC (1u << 6)

/* object types for lst_get */
enum { LST_OBJ_HIT = 0, LST_OBJ_MD = 1, LST_OBJ_LS = 2, LST_OBJ_T3 = 3, LST_OBJ_T5C = 4, LST_OBJ_T5 = 5,
       LST_OBJ_TC = 6, LST_OBJ_MATCH5 = 7, LST_OBJ_TCC = 8, LST_OBJ_TCX = 9, LST_OBJ_GRAPH = 10, LST_N_OBJ = 11 };

/* indices into counts[] of lst_status: number of objects per type after clamping to capacity,
 * then the UNCLAMPED totals (what the stage would have produced), then pair-test counts. */
enum { LST_CNT_HIT = 0, LST_CNT_MD, LST_CNT_LS, LST_CNT_T3, LST_CNT_T5C, LST_CNT_T5, LST_CNT_TC,
       LST_CNT_RAW_MD, LST_CNT_RAW_LS, LST_CNT_RAW_T3, LST_CNT_RAW_T5C, LST_CNT_RAW_T5, LST_CNT_RAW_TC,
       LST_CNT_PT5, LST_CNT_T5TC, LST_CNT_PT3, LST_CNT_PLSTC,
       /* bookkeeping of the bucketed pLS matching: first-anchor tests executed / pairs fully tested */
       LST_CNT_M5_TESTS, LST_CNT_M5_CAND, LST_CNT_M3_TESTS, LST_CNT_M3_CAND,
       /* internal: fill of the MD / LS record buffers; tile tickets of the row scans and of the T3 / T5 tiles */
       LST_CNT_FILL_MD, LST_CNT_FILL_LS, LST_CNT_TK_SENSOR, LST_CNT_TK_MD, LST_CNT_TK_LS, LST_CNT_TK_T5,
       LST_CNT_DYN_T3, LST_CNT_DYN_T5,
       /* f1: number of track candidates kept by the duplicate cleaning; tile ticket of that step (internal entries such as
        * the tickets are bookkeeping, not results; the header copy read by lst_read_tc_* carries 0 in LST_CNT_TK_TCC) */
       LST_CNT_TCC, LST_CNT_TK_TCC, LST_N_CNT = 32 };

typedef struct lst_ctx lst_ctx; /* opaque; owned by the library, freed by lst_destroy */

/* Static detector description (SPEC.md 2).  All pointers HOST; copied to the device by lst_create. */
typedef struct {
  int32_t n_modules;
  const uint8_t* subdet;      /* [n_modules] 0 barrel, 1 endcap                                   */
  const uint8_t* mtype;       /* [n_modules] 0 PS, 1 2S                                           */
  const int32_t* conn_rowptr; /* [n_modules+1] CSR of module -> connected modules, rowptr[0] = 0  */
  const int32_t* conn_col;    /* [rowptr[n_modules]] ascending and unique within a row, no self   */
  const float* dnn_weights;   /* [1857] W1[32][23], b1[32], W2[32][32], b2[32], w3[32], b3 for the default network;
                               * in general lst_dnn_n_weights(n_feat, n_hidden) floats: W1[32][n_feat], b1[32],
                               * (n_hidden - 1) x (W[32][32], b[32]), w_out[32], b_out (SPEC.md 4.9)              */
  const uint8_t* layer;       /* optional [n_modules]: detector layer of each module (1..6 barrel, 7..11 disks).  An input
                               * feature of the 38-input DNN (NULL = 0 everywhere).  When given it also selects the faster
                               * of the two exact pixel-seed prefilters of step a6 (pLS binned by where their helix
                               * crosses each layer); that choice never changes a
                               * result: any labelling, or none, gives the same matches (only the run time changes)  */
  int32_t dnn_n_feat;         /* 0 or 23: the 23 inputs of configs[0] (SPEC.md 4.5); 38: the paper's input list (4.9) */
  int32_t dnn_n_hidden;       /* 0 or 2: two hidden layers of 32; 1, 3, 4: the depth scan of PAPER.md:78 */
} lst_geometry;

/* Number of floats of `dnn_weights` for a DNN variant. */
int lst_dnn_n_weights(int32_t n_feat, int32_t n_hidden);

/* Per-slot capacities (objects).  max_tc is forced to >= max_pls + max_t5 internally. */
typedef struct {
  int32_t n_slots, max_hits, max_md, max_ls, max_t3, max_t5c, max_t5, max_pls;
} lst_caps;

/* Device view of one object list of one slot (lst_get).  Pointers are DEVICE pointers into the
 * caller's workspace, valid until lst_destroy; contents are valid after the lst_run that produced
 * them completes and until the next lst_run on that slot.  `count` is a DEVICE pointer to the
 * clamped object count.  Unused entries are NULL.  Layouts (row-major, `capacity` rows):
 *  HIT   : i0 = orig[n] int32 (sorted position -> original hit index), i1 = sensor_start[2M+1],
 *          f0 = xyzr as float4 (x, y, z, r = sqrt(x*x + y*y))
 *  MD    : i0 = hits[n][2] int32 (ORIGINAL lower, upper hit index), i1 = modt[n] int32 (module<<2 |
 *          subdet<<1 | mtype), f0 = anchor[n] float4 (x, y, z, r), f1 = cw[n] float2 (c, w),
 *          i2 = md_start[M+1]
 *  LS    : i0 = ab[n][2] int32 MD indices, f0 = c[n], i1 = ls_start[n_md+1]
 *  T3    : i0 = abc[n][4] int32 (MD a, b, c, first LS), i1 = second LS [n], f0 = k[n],
 *          i2 = t3_start[n_md+1]
 *  T5C   : i0 = md[n][5] int32, i1 = t3[n][2] int32, f0 = curv[n][3] (c_in, c_br, c_out),
 *          f1 = feat[n][n_feat] (23 or 38), f2 = score[n], i2 = pass[n] int32 (0/1)
 *  T5    : i0 = cand[n] int32 (index into T5C)
 *  TC    : i0 = tc[n][3] int32 (type 0 pT5 / 1 T5 / 2 pT3 / 3 pLS, pLS index or -1, T5-list or T3
 *          index or -1)
 *  MATCH5: i0 = best5_pls[n_t5] int32 (-1 = unmatched), f0 = chi2[n_t5]
 *  TCC   : i0 = tcc[n][3] int32: the TC rows kept by the duplicate cleaning (SPEC.md 4.7), in TC order
 *  GRAPH : the MD / LS graph of PAPER.md:127 (SPEC.md 4.8), valid after lst_export_graph: count = number of nodes (MDs);
 *          i0 = rowptr[n_md+1] (CSR over the inner MD; = ls_start), i1 = col[n_ls] (outer MD of every LS), i2 = node hits
 *          [n_md][2] (ORIGINAL lower, upper hit index), f0 = node features [n_md][8] (x, y, z, r, phi, eta, c_md, w_md),
 *          f1 = edge feature c_ls[n_ls]
 *  TCX   : per row of the TC list (count = the TC count): i0 = keep[n] int32 (1 = kept), i1 = hits[n][12] int32 (the ten ORIGINAL hit
 *          indices of the candidate's MDs, lower then upper, -1 padded, then two -1 to make rows 48 bytes), i2 = q[n] (bit pattern of the chi2 in its rank key)
 */
typedef struct {
  int32_t capacity;
  const int32_t* count;
  const int32_t* i0;
  const int32_t* i1;
  const int32_t* i2;
  const float* f0;
  const float* f1;
  const float* f2;
} lst_view;

/* Bytes of device workspace lst_create needs for these capacities.  Validates the geometry
 * (LST_EINVAL on null pointers, non-monotone rowptr, column out of range / unsorted / duplicate /
 * self-link, non-positive capacities). */
int lst_workspace_bytes(const lst_geometry* geo, const lst_caps* caps, size_t* out_bytes);

/* Build a context in `dev_workspace` (DEVICE, 256-byte aligned, >= lst_workspace_bytes) and upload
 * the geometry, CSR and DNN weights (synchronous).  The workspace must outlive the context. */
int lst_create(const lst_geometry* geo, const lst_caps* caps, void* dev_workspace, size_t bytes, lst_ctx** out);

/* Bind one event to a slot (SPEC.md 2).  DEVICE pointers; NOT copied: they must stay valid and
 * unchanged until the lst_run that consumes them has completed.  n_hits <= max_hits,
 * n_pls <= max_pls, else LST_EINVAL.  d_key[i] = 2*module + isUpper. */
int lst_load_event(lst_ctx* ctx, int32_t slot, int32_t n_hits, const float* d_x, const float* d_y,
                   const float* d_z, const uint32_t* d_key, int32_t n_pls, const float* d_px,
                   const float* d_py, const float* d_pz, const float* d_z0, const int8_t* d_q,
                   void* cuda_stream);

/* Same with HOST pointers (pinned memory recommended): enqueues the host->device copies into the
 * slot's staging area on `cuda_stream`.  Host buffers must stay valid until the copies complete.
 * The staging area is packed [x|y|z|key] and [px|py|pz|z0|q]; when the host arrays are adjacent in
 * memory in that order (h_y == h_x + n_hits, ...) each group is copied with ONE transfer. */
int lst_load_event_host(lst_ctx* ctx, int32_t slot, int32_t n_hits, const float* h_x, const float* h_y,
                        const float* h_z, const uint32_t* h_key, int32_t n_pls, const float* h_px,
                        const float* h_py, const float* h_pz, const float* h_z0, const int8_t* h_q,
                        void* cuda_stream);

/* Batched host load of slots [first_slot, first_slot + n): ONE host->device copy and one bind launch.
 * `h_blob` (HOST, pinned recommended) = int32 desc[n][2] = (n_hits, n_pls) per event, padded to a multiple of
 * 16 bytes, then per event one block padded to a multiple of 16 bytes: x[n_hits] y[n_hits] z[n_hits] (f32)
 * key[n_hits] (u32) px[n_pls] py[n_pls] pz[n_pls] z0[n_pls] (f32) q[n_pls] (i8).  `blob_bytes` = size of the
 * buffer (>= the packed size).  LST_EINVAL on sizes above the capacities or a short buffer. */
int lst_load_batch_host(lst_ctx* ctx, int32_t first_slot, int32_t n, const void* h_blob, size_t blob_bytes,
                        void* cuda_stream);

/* The same with 16-bit sensor keys (14 instead of 16 bytes per hit over the host link): per event x[n_hits] y[n_hits] z[n_hits]
 * (f32), key[n_hits] (u16, the array padded to a multiple of 4 bytes), then the pLS arrays as above; the event block padded to a
 * multiple of 16 bytes.  Needs 2 * n_modules <= 65535 (LST_EINVAL otherwise). */
int lst_load_batch_host16(lst_ctx* ctx, int32_t first_slot, int32_t n, const void* h_blob, size_t blob_bytes,
                          void* cuda_stream);

/* Batched read-back: h_out (HOST int32[n][LST_N_CNT + 3*max_rows]) receives, per slot, the counters (status word in
 * entry LST_N_CNT-1) and the first min(max_rows, count) TC rows (the rest of a slot's rows is left untouched on
 * the device side, i.e. undefined).  One pack launch + ONE device->host copy.  max_rows <= max_pls + max_t5. */
int lst_read_tc_batch_host(lst_ctx* ctx, int32_t first_slot, int32_t n, int32_t* h_out, int32_t max_rows,
                           void* cuda_stream);

/* The same with self-contained rows: h_out (HOST int32[n][LST_N_CNT + 13*max_rows]); a row is (type, pLS, object index)
 * followed by the candidate's ten ORIGINAL hit indices (SPEC.md 5: lower, upper hit of each of its MDs in order; the five
 * MDs of a pT5 / T5, the three of a pT3, -1 padded; a pLS candidate has none). */
int lst_read_tc_hits_batch_host(lst_ctx* ctx, int32_t first_slot, int32_t n, int32_t* h_out, int32_t max_rows,
                                void* cuda_stream);

/* Enqueue the whole chain a0..a6 (SPEC.md 4.0-4.6) for one slot / for slots
 * [first_slot, first_slot + n) in single batched launches (event index = a grid dimension).
 * On a capturable stream (any stream but the legacy default stream 0) the launch sequence is captured once per
 * (first_slot, n) and replayed as a CUDA graph; the environment variable LST_GRAPHS=0 (read by lst_create) keeps
 * direct launches.  Results are identical either way. */
int lst_run(lst_ctx* ctx, int32_t slot, void* cuda_stream);
int lst_run_batch(lst_ctx* ctx, int32_t first_slot, int32_t n, void* cuda_stream);

/* Device views of a slot's object lists. */
int lst_get(lst_ctx* ctx, int32_t slot, int32_t objtype, lst_view* out);

/* Synchronise `cuda_stream`, then return the slot's status bits and counts[LST_N_CNT] (HOST). */
int lst_status(lst_ctx* ctx, int32_t slot, uint32_t* status_bits, int32_t* counts, void* cuda_stream);

/* Enqueue device->host copies of the slot's counters (HOST int32[LST_N_CNT], then status word in
 * h_counts[LST_N_CNT-1]) and of the first `max_rows` rows of its TC list (HOST int32[max_rows][3]). */
/* When h_tc == h_counts + LST_N_CNT (one host buffer) both are read with ONE transfer. */
int lst_read_tc_host(lst_ctx* ctx, int32_t slot, int32_t* h_counts, int32_t* h_tc, int32_t max_rows,
                     void* cuda_stream);

/* Number of kernel launches one lst_run / lst_run_batch enqueues (for the harness' accounting). */
int lst_launches_per_run(void);

/* Profiling variant of lst_run_batch: same launches with a CUDA event recorded on `cuda_stream`
 * between them; synchronises, then writes the device time in ms of the memset pair and of each of
 * the lst_launches_per_run() kernels to h_ms[0 .. lst_launches_per_run()] (HOST).  Not a bench
 * path: the events serialise nothing but add launch gaps. */
int lst_run_batch_profile(lst_ctx* ctx, int32_t first_slot, int32_t n, void* cuda_stream, float* h_ms);

/* f4: pack the MD / LS graph (nodes = MDs, edges = LSs, SPEC.md 4.8) of slots [first_slot, first_slot + n)
 * after their lst_run: ONE launch that writes the node-feature table and the CSR column array into the workspace; the row
 * pointer, the node -> original-hit table and the edge feature are the chain's own MD / LS outputs.  Read the result through
 * lst_get(LST_OBJ_GRAPH).  Enqueues only. */
int lst_export_graph(lst_ctx* ctx, int32_t first_slot, int32_t n, void* cuda_stream);

/* Measurement only: sustained fp32 throughput of this GPU in Tflop/s (HOST *h_tflops), counted as one multiply + one add
 * per chain step, with separately rounded multiply and add (fused = 0: the form the cut arithmetic must use) or with fused
 * multiply-add (fused = 1: allowed in the DNN).  Runs a few ms of a register-only kernel on `cuda_stream` and synchronises.
 * These are the denominators of the ALU-bound rooflines in bench.py. */
int lst_measure_fp32(lst_ctx* ctx, int32_t fused, float* h_tflops, void* cuda_stream);

/* Name of entry i of h_ms ("memset", "a0.hist", ... , "a6.tc_emit"); NULL when out of range. */
const char* lst_launch_name(int32_t i);

void lst_destroy(lst_ctx* ctx);

/* ---- a0 without a workspace: for callers that cannot allocate device memory ------------------------------------------
 * Every call above works in a workspace the caller allocates and hands to lst_create.  Some callers cannot do even
 * that: a plugin inside a trigger / event-processing job whose framework gave out all device memory at start-up and
 * passes a module its input and output buffers and nothing more, or an event loop where cudaMalloc / cudaFree are
 * forbidden because they synchronise the whole device and take an unbounded time.  For them this ONE entry point runs
 * the hit ingest of step a0 (SPEC.md 4.0; hits grouped by pT-module sensor) with no context, no workspace
 * and no allocation of any kind: its temporaries sit in a fixed array built into the library
 * (LST_STATIC_SCRATCH_BYTES, about 1.3 MB, held by every GPU that loads the library until the process exits).
 *
 *  in  (DEVICE): d_x, d_y, d_z [n_hits] float; d_key [n_hits] uint32 = 2*module + isUpper
 *  out (DEVICE): d_hit_xyzr [n_hits][4] float (16-byte aligned): hits in sensor order, stable in the original index,
 *                as (x, y, z, r = sqrt(x*x + y*y)); d_hit_orig [n_hits] int32: sorted position -> original index;
 *                d_sensor_start [2*n_modules + 1] int32: first sorted position of each sensor, last entry = hits kept;
 *                d_count [2] int32: hits kept, status bits (LST_ST_BAD_KEY if a key >= 2*n_modules was dropped).
 *                Rows past "hits kept" are left untouched.  Same values as lst_get(LST_OBJ_HIT) after lst_run.
 *  Limits      : n_hits <= LST_STATIC_MAX_HITS and n_modules <= LST_STATIC_MAX_MODULES, else LST_ETOOBIG and nothing is
 *                enqueued.  LST_EINVAL on null / misaligned pointers or negative sizes, LST_ECUDA if a CUDA call fails.
 *  Device      : the device that owns `cuda_stream` and the buffers must be the current device.  The first call on each
 *                device also looks up where the built-in array lives on that device (a one-time set-up that must not
 *                happen inside a stream capture: make the first call on a device before any capture starts).
 *  Sharing     : all calls on one GPU use the same array.  Each call clears the counters it needs, so a call never sees
 *                the previous one's data, but two calls that run on the GPU at the same time (two streams, two host
 *                threads) corrupt each other: keep them on one stream or order them with an event.
 *  Enqueues only (one memset and four small kernels on `cuda_stream`); no host synchronisation. */
#define LST_STATIC_MAX_HITS 131072
#define LST_STATIC_MAX_MODULES 32768
#define LST_STATIC_SCRATCH_BYTES (4 * (128 + 2 * LST_STATIC_MAX_MODULES + 2 * LST_STATIC_MAX_HITS))
int lst_sort_hits_static(int32_t n_hits, int32_t n_modules, const float* d_x, const float* d_y, const float* d_z,
                         const uint32_t* d_key, float* d_hit_xyzr, int32_t* d_hit_orig, int32_t* d_sensor_start,
                         int32_t* d_count, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* LST_H_ */
