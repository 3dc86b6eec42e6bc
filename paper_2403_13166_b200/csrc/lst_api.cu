// lst_api.cu -- the C ABI of include/lst.h: workspace carving, geometry upload, launch sequence.
// Host logic only; every step of the hot path runs in the kernels of lst_kernels.cuh.
#include <cuda_runtime.h>
#include <new>
#include <cstdlib>
#include <map>
#include <vector>
#include "lst_tuples.cuh"

using namespace lst;

struct lst_ctx {
  int n_slots = 0;
  int n_modules = 0;
  Geo geo{};
  Caps caps{};
  Slot* d_slots = nullptr;        // device array [n_slots]
  std::vector<Slot> h_slots;      // host mirror of the carved pointers (inputs not tracked)
  char* batch_in = nullptr; size_t batch_in_stride = 0;     // staging of lst_load_batch_host, one stride per slot
  int* batch_out = nullptr; size_t batch_out_stride = 0;    // staging of lst_read_tc_batch_host (ints per slot)
  char* zero_base = nullptr; size_t zero_stride = 0;
  char* ones_base = nullptr; size_t ones_stride = 0;
  bool sticky_cuda_error = false;
  int n_sm = 148;                 // multiprocessors of the context's device (queried by lst_create): sizes every grid
  bool capturing = false;         // run_sequence is being recorded into a graph
  bool use_xs = true;             // a6 with per-surface crossing keys when the geometry carries layers (LST_XS=0: the generic (h, zeta, psi) buckets)
  bool use_pdl = false;           // programmatic dependent launch between the kernels of the chain (LST_PDL=1 enables; measured: no gain under graph replay)
  bool use_graphs = true;         // replay lst_run_batch as a CUDA graph on capturable streams (LST_GRAPHS=0 disables)
  std::map<long long, cudaGraphExec_t> graphs;   // (first_slot, n) -> instantiated launch sequence
  cudaStream_t side = nullptr;                   // capture-time side branch (pLS binning runs beside a0..a5)
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
};

#ifndef LS_GRID_PER_SM
#define LS_GRID_PER_SM 7
#endif
namespace {

constexpr size_t ALIGN = 256;
inline size_t up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Carver {   // walks the workspace; with base == nullptr it only measures
  char* base; size_t off = 0;
  template <typename T> T* take(size_t n) {
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += up(n * sizeof(T));
    return p;
  }
};

int validate(const lst_geometry* g, const lst_caps* c) {
  if (!g || !c || !g->subdet || !g->mtype || !g->conn_rowptr || !g->conn_col || !g->dnn_weights) return LST_EINVAL;
  if (g->n_modules <= 0 || g->n_modules > (1 << 28)) return LST_EINVAL;
  if (c->n_slots <= 0 || c->max_hits <= 0 || c->max_md <= 0 || c->max_ls <= 0 || c->max_t3 <= 0 || c->max_t5c <= 0 ||
      c->max_t5 <= 0 || c->max_pls <= 0)
    return LST_EINVAL;
  if (c->max_pls > (1 << 28) / 5) return LST_EINVAL;
  if (g->dnn_n_feat != 0 && g->dnn_n_feat != N_FEAT && g->dnn_n_feat != N_FEAT_MAX) return LST_EINVAL;
  if (g->dnn_n_hidden < 0 || g->dnn_n_hidden > 4) return LST_EINVAL;
  const int M = g->n_modules;
  if (g->conn_rowptr[0] != 0) return LST_EINVAL;
  for (int m = 0; m < M; ++m) {
    const int b = g->conn_rowptr[m], e = g->conn_rowptr[m + 1];
    if (e < b) return LST_EINVAL;
    for (int i = b; i < e; ++i) {
      const int col = g->conn_col[i];
      if (col < 0 || col >= M || col == m) return LST_EINVAL;
      if (i > b && g->conn_col[i - 1] >= col) return LST_EINVAL;
    }
    if (g->subdet[m] > 1 || g->mtype[m] > 1) return LST_EINVAL;
  }
  return LST_OK;
}

Caps make_caps(const lst_caps* c) {
  Caps k;
  k.max_hits = c->max_hits; k.max_md = c->max_md; k.max_ls = c->max_ls; k.max_t3 = c->max_t3;
  k.max_t5c = c->max_t5c; k.max_t5 = c->max_t5; k.max_pls = c->max_pls; k.max_tc = c->max_pls + c->max_t5;
  return k;
}

// One pass lays out the whole workspace; used both to measure and to carve.
struct Layout {
  char* batch_in; size_t batch_in_stride; int* batch_out; size_t batch_out_stride;
  Slot* slots; uint8_t* modt; uint8_t* layer; uint8_t* xs_layer; int* rowptr; int* col; float* weights; int* run_ptr; int* run_c0; int* run_c1;
  char* zero_base; size_t zero_stride; char* ones_base; size_t ones_stride;
  size_t total;
};

Layout lay_out(char* base, int M, int nnz, const Caps& k, int n_slots, std::vector<Slot>* out) {
  Carver cv{base};
  Layout L{};
  L.slots = cv.take<Slot>(n_slots);
  L.modt = cv.take<uint8_t>(M);
  L.layer = cv.take<uint8_t>(M);
  L.xs_layer = cv.take<uint8_t>(M);
  L.rowptr = cv.take<int>(M + 1);
  L.col = cv.take<int>(nnz > 0 ? nnz : 1);
  L.weights = cv.take<float>(dnn_n_weights(N_FEAT_MAX, 4));
  L.run_ptr = cv.take<int>(M + 1);
  L.run_c0 = cv.take<int>(nnz > 0 ? nnz : 1);      // a row has at most as many runs as entries
  L.run_c1 = cv.take<int>(nnz > 0 ? nnz : 1);
  L.batch_in_stride = blob_event_bytes(k.max_hits, k.max_pls) + 16;
  L.batch_in = cv.take<char>(L.batch_in_stride * n_slots + 1024);
  L.batch_out_stride = LST_N_CNT + 13 * (size_t)k.max_tc;
  L.batch_out = cv.take<int>(L.batch_out_stride * n_slots);
  if (out) out->assign(n_slots, Slot{});
  // zero region (contiguous over slots so one memset covers a batch)
  {
    Carver z{nullptr};
    z.take<int>(LST_N_CNT); z.take<int>(2 * M + 2); z.take<int>(N_TK); z.take<unsigned>(XS_NS); z.take<unsigned>(XS_NS);
    L.zero_stride = z.off;
    L.zero_base = base ? base + cv.off : nullptr;
    for (int s = 0; s < n_slots; ++s) {
      Carver c2{base ? base + cv.off + s * L.zero_stride : nullptr};
      int* cnt = c2.take<int>(LST_N_CNT);
      int* ss = c2.take<int>(2 * M + 2);
      int* tk = c2.take<int>(N_TK);
      unsigned* shi = c2.take<unsigned>(XS_NS);
      unsigned* srh = c2.take<unsigned>(XS_NS);
      if (out) { (*out)[s].cnt = cnt; (*out)[s].sensor_start = ss; (*out)[s].tk = tk; (*out)[s].surf_hi = shi; (*out)[s].surf_rhi = srh; }
    }
    cv.off += L.zero_stride * n_slots;
  }
  // 0xFF region
  {
    Carver z{nullptr};
    z.take<unsigned long long>(k.max_pls); z.take<unsigned long long>(k.max_pls); z.take<int>(k.max_md); z.take<int>(k.max_hits); z.take<unsigned>(XS_NS);
    L.ones_stride = z.off;
    L.ones_base = base ? base + cv.off : nullptr;
    for (int s = 0; s < n_slots; ++s) {
      Carver c2{base ? base + cv.off + s * L.ones_stride : nullptr};
      auto* w5 = c2.take<unsigned long long>(k.max_pls);
      auto* w3 = c2.take<unsigned long long>(k.max_pls);
      int* head = c2.take<int>(k.max_md);
      int* hhead = c2.take<int>(k.max_hits);
      unsigned* slo = c2.take<unsigned>(XS_NS);
      if (out) { (*out)[s].win5 = w5; (*out)[s].win3 = w3; (*out)[s].md_head = head; (*out)[s].hit_head = hhead; (*out)[s].surf_lo = slo; }
    }
    cv.off += L.ones_stride * n_slots;
  }
  for (int s = 0; s < n_slots; ++s) {
    Slot t{};
    t.epoch_dev = cv.take<unsigned>(4); t.tmp_a = cv.take<float4>(k.max_hits); t.tmp_k = cv.take<int>(k.max_hits); t.hit = cv.take<float4>(k.max_hits); t.hit_orig = cv.take<int>(k.max_hits);
    t.md_rec = cv.take<MdRec>(k.max_md);
    t.md_hits = cv.take<int2>(k.max_md); t.md_modt = cv.take<int>(k.max_md);
    t.md_pos = cv.take<float4>(k.max_md); t.md_cw = cv.take<float2>(k.max_md); t.md_aux = cv.take<float4>(k.max_md); t.md_start = cv.take<int>(M + 8);
    t.ls_rec = cv.take<LsRec>(k.max_ls);
    t.ls_tab = cv.take<int>(16 * (size_t)M); t.ls_start = cv.take<int>(k.max_md + 8); t.ls_ab = cv.take<int2>(k.max_ls); t.ls_c = cv.take<float>(k.max_ls);
    t.chain_sensor = cv.take<unsigned long long>(2 * (size_t)M / SCAN_TILE + 4); t.chain_md = cv.take<unsigned long long>(M / SCAN_TILE + 4);
    t.chain_ls = cv.take<unsigned long long>(k.max_md / SCAN_TILE + 4); t.chain_t5s = cv.take<unsigned long long>(k.max_t5c / 128 + 4);
    t.chain_t3 = cv.take<unsigned long long>(k.max_ls / TUPLE_TPB + 4); t.chain_t5 = cv.take<unsigned long long>(k.max_t3 / TUPLE_TPB + 4);
    t.t3_off = cv.take<int>(k.max_ls + 8); t.t3_abc = cv.take<int4>(k.max_t3); t.t3_l1 = cv.take<int>(k.max_t3);
    t.t3_k = cv.take<float>(k.max_t3); t.t3_start = cv.take<int>(k.max_md + 8);
    t.t5_off = cv.take<int>(k.max_t3 + 8); t.t5c_md = cv.take<int>(5 * (size_t)k.max_t5c); t.t5c_t3 = cv.take<int2>(k.max_t5c);
    t.t5c_curv = cv.take<float>(3 * (size_t)k.max_t5c); t.t5c_feat = cv.take<float>((size_t)N_FEAT_MAX * k.max_t5c);
    t.t5c_score = cv.take<float>(k.max_t5c); t.t5c_pass = cv.take<int>(k.max_t5c);
    t.t5_list = cv.take<int>(k.max_t5);
    t.pls_a = cv.take<float4>(k.max_pls); t.pls_b = cv.take<float2>(k.max_pls); t.pls_key = cv.take<int>(k.max_pls);
    t.pls_sa = cv.take<float4>(k.max_pls); t.pls_sb = cv.take<float2>(k.max_pls); t.pls_sidx = cv.take<int>(k.max_pls); t.pls_pos = cv.take<int>(k.max_pls); t.pls_taken = cv.take<int>(k.max_pls);
    t.pls_bin_start = cv.take<int>(PLS_NBINS + 1); t.xs_key = cv.take<int>((size_t)XS_NS * k.max_pls); t.xs_start = cv.take<int>((size_t)XS_NS * (XS_BINS + 1)); t.xs_ent = cv.take<float4>((size_t)XS_NS * 2 * k.max_pls); t.best5 = cv.take<int>(k.max_t5);
    t.chi5 = cv.take<float>(k.max_t5); t.pt5_next = cv.take<int>(5 * (size_t)k.max_pls); t.best3 = cv.take<int>(k.max_t3);
    t.chi3 = cv.take<float>(k.max_t3); t.tc_hdr = cv.take<int>(LST_N_CNT + 3 * (size_t)k.max_tc); t.tc = t.tc_hdr ? t.tc_hdr + LST_N_CNT : nullptr;
    t.tc_hits = cv.take<int>(TC_HSTRIDE * (size_t)k.max_tc); t.tc_q = cv.take<int>(k.max_tc); t.tc_next = cv.take<int>(10 * (size_t)k.max_tc); t.tc_keep = cv.take<int>(k.max_tc); t.tc_sig = cv.take<unsigned long long>(k.max_tc); t.chain_tce = cv.take<unsigned long long>((3 * (size_t)k.max_pls + k.max_t5) / TCE_TPB + 4);
    t.tcc = cv.take<int>(3 * (size_t)k.max_tc); t.chain_tcc = cv.take<unsigned long long>(k.max_tc / TCC_ROWS + 4);
    t.g_node = cv.take<float>(8 * (size_t)k.max_md); t.g_col = cv.take<int>(k.max_ls);
    t.st_hits = cv.take<float>(4 * (size_t)k.max_hits); t.st_pls = cv.take<float>(5 * (size_t)k.max_pls);
    if (out) {
      Slot& d = (*out)[s];
      t.cnt = d.cnt; t.sensor_start = d.sensor_start; t.tk = d.tk; t.surf_hi = d.surf_hi; t.surf_rhi = d.surf_rhi; t.surf_lo = d.surf_lo; t.win5 = d.win5; t.win3 = d.win3; t.md_head = d.md_head; t.hit_head = d.hit_head;
      d = t;
    }
  }
  L.total = cv.off;
  return L;
}

// launch with (or without) programmatic stream serialization, see pdl_begin().  The first launch error of a sequence is kept
// in t_launch_err (run_sequence clears it on entry and reports it on exit).
thread_local cudaError_t t_launch_err = cudaSuccess;
template <typename... KArgs, typename... Args>
inline void launch(bool pdl, void (*k)(KArgs...), dim3 g, dim3 b, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = g; cfg.blockDim = b; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, k, static_cast<KArgs>(args)...);
  if (e != cudaSuccess && t_launch_err == cudaSuccess) t_launch_err = e;
}

inline bool bad(lst_ctx* c, cudaError_t e) {
  if (e != cudaSuccess) { c->sticky_cuda_error = true; return true; }
  return false;
}

constexpr int N_LAUNCHES = 19;   // kernels per lst_run / lst_run_batch (plus two memsets)

}  // namespace

extern "C" {

int lst_launches_per_run(void) { return N_LAUNCHES; }

int lst_dnn_n_weights(int32_t n_feat, int32_t n_hidden) {
  if ((n_feat != N_FEAT && n_feat != N_FEAT_MAX) || n_hidden < 1 || n_hidden > 4) return LST_EINVAL;
  return dnn_n_weights(n_feat, n_hidden);
}

int lst_workspace_bytes(const lst_geometry* geo, const lst_caps* caps, size_t* out_bytes) {
  if (!out_bytes) return LST_EINVAL;
  const int rc = validate(geo, caps);
  if (rc != LST_OK) return rc;
  const Caps k = make_caps(caps);
  const Layout L = lay_out(nullptr, geo->n_modules, geo->conn_rowptr[geo->n_modules], k, caps->n_slots, nullptr);
  *out_bytes = L.total;
  return LST_OK;
}

int lst_create(const lst_geometry* geo, const lst_caps* caps, void* dev_workspace, size_t bytes, lst_ctx** out) {
  if (!out || !dev_workspace) return LST_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev_workspace) % ALIGN) return LST_EINVAL;
  const int rc = validate(geo, caps);
  if (rc != LST_OK) return rc;
  lst_ctx* c = new (std::nothrow) lst_ctx();
  if (!c) return LST_ENOMEM;
  const int M = geo->n_modules, nnz = geo->conn_rowptr[M];
  c->caps = make_caps(caps);
  c->n_slots = caps->n_slots;
  c->n_modules = M;
  const Layout L = lay_out(static_cast<char*>(dev_workspace), M, nnz, c->caps, c->n_slots, &c->h_slots);
  if (L.total > bytes) { delete c; return LST_ENOMEM; }
  c->d_slots = L.slots;
  c->zero_base = L.zero_base; c->zero_stride = L.zero_stride;
  c->batch_in = L.batch_in; c->batch_in_stride = L.batch_in_stride; c->batch_out = L.batch_out; c->batch_out_stride = L.batch_out_stride;
  c->ones_base = L.ones_base; c->ones_stride = L.ones_stride;
  std::vector<uint8_t> modt(M);
  for (int m = 0; m < M; ++m) modt[m] = uint8_t((geo->subdet[m] << 1) | geo->mtype[m]);
  cudaError_t e = cudaMemcpy(L.modt, modt.data(), M, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(L.rowptr, geo->conn_rowptr, sizeof(int) * (M + 1), cudaMemcpyHostToDevice);
  if (e == cudaSuccess && nnz > 0) e = cudaMemcpy(L.col, geo->conn_col, sizeof(int) * nnz, cudaMemcpyHostToDevice);
  const int n_feat = geo->dnn_n_feat ? geo->dnn_n_feat : N_FEAT, n_hidden = geo->dnn_n_hidden ? geo->dnn_n_hidden : 2;
  if (e == cudaSuccess) e = cudaMemcpy(L.weights, geo->dnn_weights, sizeof(float) * dnn_n_weights(n_feat, n_hidden), cudaMemcpyHostToDevice);
  {
    std::vector<uint8_t> lay(M, 0);
    if (geo->layer) for (int m = 0; m < M; ++m) lay[m] = geo->layer[m];
    if (e == cudaSuccess) e = cudaMemcpy(L.layer, lay.data(), M, cudaMemcpyHostToDevice);
    // a T3 / T5 starts on module m only if the CSR has a two-step path m -> m' -> m'': only those modules' MDs define the a6 surfaces.
    // The table holds the label reduced to the bits xs_surface() uses (<= 15), so the "not a start module" mark 255 can never
    // collide with a caller's label (any uint8, 255 included, is a legal label).
    std::vector<uint8_t> xs(M, 255);
    for (int m = 0; m < M; ++m)
      for (int i = geo->conn_rowptr[m]; i < geo->conn_rowptr[m + 1] && xs[m] == 255; ++i) {
        const int m1 = geo->conn_col[i];
        if (geo->conn_rowptr[m1 + 1] > geo->conn_rowptr[m1]) xs[m] = lay[m] & 15;
      }
    if (e == cudaSuccess) e = cudaMemcpy(L.xs_layer, xs.data(), M, cudaMemcpyHostToDevice);
  }
  {   // CSR rows -> runs of consecutive module ids (one run = one contiguous MD range, lst_pairs.cuh)
    std::vector<int> run_ptr(M + 1, 0), c0, c1;
    for (int m = 0; m < M; ++m) {
      for (int i = geo->conn_rowptr[m]; i < geo->conn_rowptr[m + 1]; ++i) {
        const int col = geo->conn_col[i];
        if (i > geo->conn_rowptr[m] && c1.back() == col) c1.back() = col + 1;
        else { c0.push_back(col); c1.push_back(col + 1); }
      }
      run_ptr[m + 1] = (int)c0.size();
    }
    if (e == cudaSuccess) e = cudaMemcpy(L.run_ptr, run_ptr.data(), sizeof(int) * (M + 1), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && !c0.empty()) e = cudaMemcpy(L.run_c0, c0.data(), sizeof(int) * c0.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && !c0.empty()) e = cudaMemcpy(L.run_c1, c1.data(), sizeof(int) * c1.size(), cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess) e = cudaMemcpy(L.slots, c->h_slots.data(), sizeof(Slot) * c->n_slots, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(c->zero_base, 0, c->zero_stride * c->n_slots);
  for (int i = 0; i < c->n_slots && e == cudaSuccess; ++i) {   // status words start at epoch 0 (never a run's epoch)
    e = cudaMemset(c->h_slots[i].epoch_dev, 0, 16);
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_sensor, 0, sizeof(unsigned long long) * (2 * (size_t)M / SCAN_TILE + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_md, 0, sizeof(unsigned long long) * (M / SCAN_TILE + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_ls, 0, sizeof(unsigned long long) * (c->caps.max_md / SCAN_TILE + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_t5s, 0, sizeof(unsigned long long) * (c->caps.max_t5c / 128 + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_tce, 0, sizeof(unsigned long long) * ((3 * (size_t)c->caps.max_pls + c->caps.max_t5) / TCE_TPB + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_tcc, 0, sizeof(unsigned long long) * (c->caps.max_tc / TCC_ROWS + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_t3, 0, sizeof(unsigned long long) * (c->caps.max_ls / TUPLE_TPB + 4));
    if (e == cudaSuccess) e = cudaMemset(c->h_slots[i].chain_t5, 0, sizeof(unsigned long long) * (c->caps.max_t3 / TUPLE_TPB + 4));
  }
  if (e == cudaSuccess) e = cudaDeviceSynchronize();       // the memsets above are asynchronous on device memory
  if (e == cudaSuccess) {
    int dev = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess && c->n_sm <= 0) e = cudaErrorInvalidDevice;
  }
  if (e != cudaSuccess) { delete c; return LST_ECUDA; }
  if (cudaFuncSetAttribute(k_pls_bin, cudaFuncAttributeMaxDynamicSharedMemorySize, PLS_BIN_SMEM) != cudaSuccess) { delete c; return LST_ECUDA; }
  if (const char* g = std::getenv("LST_GRAPHS")) c->use_graphs = !(g[0] == '0');
  if (const char* g = std::getenv("LST_PDL")) c->use_pdl = !(g[0] == '0');
  if (const char* g = std::getenv("LST_XS")) c->use_xs = !(g[0] == '0');
  if (c->use_graphs) {            // host-side objects only; without them the binning simply stays in line
    if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess) c->side = nullptr;
    if (c->side && (cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                    cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess)) {
      cudaStreamDestroy(c->side); c->side = nullptr;
    }
    (void)cudaGetLastError();
  }
  c->geo.n_modules = M; c->geo.modt = L.modt; c->geo.rowptr = L.rowptr; c->geo.col = L.col; c->geo.weights = L.weights; c->geo.layer = L.layer; c->geo.xs_layer = L.xs_layer; c->geo.has_layer = (geo->layer && c->use_xs) ? 1 : 0; c->geo.n_feat = n_feat; c->geo.n_hidden = n_hidden;
  c->geo.run_ptr = L.run_ptr; c->geo.run_c0 = L.run_c0; c->geo.run_c1 = L.run_c1;
  *out = c;
  return LST_OK;
}

int lst_load_event(lst_ctx* c, int32_t slot, int32_t n_hits, const float* d_x, const float* d_y, const float* d_z,
                   const uint32_t* d_key, int32_t n_pls, const float* d_px, const float* d_py, const float* d_pz,
                   const float* d_z0, const int8_t* d_q, void* cuda_stream) {
  if (!c || slot < 0 || slot >= c->n_slots || n_hits < 0 || n_pls < 0) return LST_EINVAL;
  if (n_hits > c->caps.max_hits || n_pls > c->caps.max_pls) return LST_EINVAL;
  if (n_hits > 0 && (!d_x || !d_y || !d_z || !d_key)) return LST_EINVAL;
  if (n_pls > 0 && (!d_px || !d_py || !d_pz || !d_z0 || !d_q)) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  k_bind<<<1, 1, 0, static_cast<cudaStream_t>(cuda_stream)>>>(c->d_slots, slot, d_x, d_y, d_z, d_key, n_hits, d_px, d_py,
                                                               d_pz, d_z0, d_q, n_pls);
  return bad(c, cudaGetLastError()) ? LST_ECUDA : LST_OK;
}

int lst_load_event_host(lst_ctx* c, int32_t slot, int32_t n_hits, const float* h_x, const float* h_y, const float* h_z,
                        const uint32_t* h_key, int32_t n_pls, const float* h_px, const float* h_py, const float* h_pz,
                        const float* h_z0, const int8_t* h_q, void* cuda_stream) {
  if (!c || slot < 0 || slot >= c->n_slots || n_hits < 0 || n_pls < 0) return LST_EINVAL;
  if (n_hits > c->caps.max_hits || n_pls > c->caps.max_pls) return LST_EINVAL;
  if (n_hits > 0 && (!h_x || !h_y || !h_z || !h_key)) return LST_EINVAL;
  if (n_pls > 0 && (!h_px || !h_py || !h_pz || !h_z0 || !h_q)) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const Slot& s = c->h_slots[slot];
  cudaError_t e = cudaSuccess;
  auto cp = [&](void* dst, const void* src, size_t n) {
    if (e == cudaSuccess && n) e = cudaMemcpyAsync(dst, src, n, cudaMemcpyHostToDevice, st);
  };
  // device staging is packed [x|y|z|key] and [px|py|pz|z0|q]; a host event packed the same way goes over in
  // two copies instead of nine
  float* dx = s.st_hits; float* dy = dx + n_hits; float* dz = dy + n_hits; uint32_t* dk = reinterpret_cast<uint32_t*>(dz + n_hits);
  float* dpx = s.st_pls; float* dpy = dpx + n_pls; float* dpz = dpy + n_pls; float* dz0 = dpz + n_pls; int8_t* dq = reinterpret_cast<int8_t*>(dz0 + n_pls);
  if (h_y == h_x + n_hits && h_z == h_y + n_hits && reinterpret_cast<const float*>(h_key) == h_z + n_hits) cp(dx, h_x, 16 * (size_t)n_hits);
  else { cp(dx, h_x, 4 * (size_t)n_hits); cp(dy, h_y, 4 * (size_t)n_hits); cp(dz, h_z, 4 * (size_t)n_hits); cp(dk, h_key, 4 * (size_t)n_hits); }
  if (h_py == h_px + n_pls && h_pz == h_py + n_pls && h_z0 == h_pz + n_pls && reinterpret_cast<const float*>(h_q) == h_z0 + n_pls) cp(dpx, h_px, 17 * (size_t)n_pls);
  else { cp(dpx, h_px, 4 * (size_t)n_pls); cp(dpy, h_py, 4 * (size_t)n_pls); cp(dpz, h_pz, 4 * (size_t)n_pls); cp(dz0, h_z0, 4 * (size_t)n_pls); cp(dq, h_q, n_pls); }
  if (bad(c, e)) return LST_ECUDA;
  return lst_load_event(c, slot, n_hits, dx, dy, dz, dk, n_pls, dpx, dpy, dpz, dz0, dq, cuda_stream);
}

// The launch sequence of one pass over slots [first, first+n).  With `ev` != nullptr an event is
// recorded before the first and after every launch (profiling entry point only).
static int run_sequence(lst_ctx* c, int32_t first, int32_t n, cudaStream_t st, cudaEvent_t* ev) {
  const Slot* sl = c->d_slots + first;
  const Geo g = c->geo;
  const Caps k = c->caps;
  int li = 0;
  t_launch_err = cudaSuccess;
#define LST_MARK() do { if (ev && bad(c, cudaEventRecord(ev[li], st))) return LST_ECUDA; ++li; } while (0)
  LST_MARK();
  if (bad(c, cudaMemsetAsync(c->zero_base + first * c->zero_stride, 0, c->zero_stride * n, st))) return LST_ECUDA;
  if (bad(c, cudaMemsetAsync(c->ones_base + first * c->ones_stride, 0xFF, c->ones_stride * n, st))) return LST_ECUDA;
  LST_MARK();
  // x-extent of the grids: enough blocks to fill the SMs (148 on a B200) several times over across the whole batch
  const int n_sm = c->n_sm;
  int gx = (n_sm * 8 + n - 1) / n;
  if (gx < 8) gx = 8;
  if (gx > 4 * n_sm) gx = 4 * n_sm;
  const dim3 G(gx, n), G1(1, n), GL(2 * gx, n);   // GL: the 128-thread link kernels
  const dim3 GS(gx < 16 ? gx : 16, n);            // look-back scans: tiles of 2048 entries by ticket
  // the pLS binning depends on the inputs only: under stream capture it becomes a side branch of the graph
  // (with a layer per module the binning uses the surfaces measured by k_md_finish: the branch forks after that kernel)
  const bool fork = c->capturing && c->side;
  const bool xs = g.has_layer != 0;
  const dim3 GX(XS_NS, n);
  if (fork && !xs) {
    if (bad(c, cudaEventRecord(c->ev_fork, st)) || bad(c, cudaStreamWaitEvent(c->side, c->ev_fork, 0))) return LST_ECUDA;
    k_pls_bin<<<G1, 1024, PLS_BIN_SMEM, c->side>>>(sl);
    if (bad(c, cudaEventRecord(c->ev_join, c->side))) return LST_ECUDA;
  }
  // every kernel after the first waits for its predecessor with griddepcontrol.wait, so its launch may overlap the
  // predecessor's tail; not under the profiling entry point (events between launches) and not across the side-branch join
  const bool pdl = c->use_pdl && !ev;
  const dim3 B128(128), B256(256), BS(SCAN_TPB), BP(PAIR_WARPS * 32), BT(TUPLE_TPB), BM(MATCH_WARPS * 32);
  launch(false, k_hist, G, B256, 0, st, sl, g); LST_MARK();
  launch(pdl, k_scan_lb<SCAN_SENSOR>, GS, BS, 0, st, sl, g, k); LST_MARK();
  launch(pdl, k_scatter, G, B256, 0, st, sl, g); LST_MARK();
  launch(pdl, k_rank, G, B256, 0, st, sl); LST_MARK();
  launch(pdl, k_md_sweep, GL, BP, 0, st, sl, g, k); LST_MARK();
  launch(pdl, k_scan_lb<SCAN_MDROW>, GS, BS, 0, st, sl, g, k); LST_MARK();
  launch(pdl, k_md_finish, GL, BP, 0, st, sl, g, k); LST_MARK();
  if (fork && xs) {
    if (bad(c, cudaEventRecord(c->ev_fork, st)) || bad(c, cudaStreamWaitEvent(c->side, c->ev_fork, 0))) return LST_ECUDA;
    k_pls_cross<<<GX, XS_TPB, XS_SMEM, c->side>>>(sl, k.max_pls);
    if (bad(c, cudaEventRecord(c->ev_join, c->side))) return LST_ECUDA;
  }
  launch(pdl, k_ls_sweep, dim3(n < 8 ? n_sm * 4 : n_sm * LS_GRID_PER_SM, (n + 31) / 32), BP, 0, st, sl, (int)n, g, k); LST_MARK();      // persistent grid: the resident blocks
  launch(pdl, k_scan_lb<SCAN_LSROW>, GS, BS, 0, st, sl, g, k); LST_MARK();
  launch(pdl, k_ls_finish, GL, BP, 0, st, sl, g, k); LST_MARK();
  launch(pdl, k_t3_one, GL, BT, 0, st, sl, k); LST_MARK();
  launch(pdl, k_t5_one, GL, BT, 0, st, sl, k); LST_MARK();
  {
#define LST_DNN(NI, NH_) launch(pdl, k_dnn<NI, NH_>, G, B128, 0, st, sl, g, k.max_t5)
    const int nh = g.n_hidden;
    if (g.n_feat == N_FEAT) { if (nh == 1) LST_DNN(N_FEAT, 1); else if (nh == 2) LST_DNN(N_FEAT, 2); else if (nh == 3) LST_DNN(N_FEAT, 3); else LST_DNN(N_FEAT, 4); }
    else { if (nh == 1) LST_DNN(N_FEAT_MAX, 1); else if (nh == 2) LST_DNN(N_FEAT_MAX, 2); else if (nh == 3) LST_DNN(N_FEAT_MAX, 3); else LST_DNN(N_FEAT_MAX, 4); }
#undef LST_DNN
  }
  LST_MARK();
  if (fork) { if (bad(c, cudaStreamWaitEvent(st, c->ev_join, 0))) return LST_ECUDA; }
  else if (xs) launch(false, k_pls_cross, GX, dim3(XS_TPB), XS_SMEM, st, sl, k.max_pls);
  else launch(false, k_pls_bin, G1, dim3(1024), PLS_BIN_SMEM, st, sl);
  LST_MARK();
  if (xs) launch(pdl && !fork, k_match<5, false, true>, G, BM, 0, st, sl, g, k.max_pls); else launch(pdl && !fork, k_match<5, false, false>, G, BM, 0, st, sl, g, k.max_pls);
  LST_MARK();
  launch(pdl, k_pt5_lists, G, B128, 0, st, sl); LST_MARK();
  if (xs) launch(pdl, k_match<3, true, true>, G, BM, 0, st, sl, g, k.max_pls); else launch(pdl, k_match<3, true, false>, G, BM, 0, st, sl, g, k.max_pls);
  LST_MARK();
  launch(pdl, k_tc_emit, dim3(gx < 48 ? gx : 48, n), dim3(TCE_TPB), 0, st, sl, k); LST_MARK();
  launch(pdl, k_tc_clean, GL, dim3(TCC_TPB), 0, st, sl, k); LST_MARK();
#undef LST_MARK
  if (li != N_LAUNCHES + 2) return LST_EINVAL;
  if (bad(c, t_launch_err)) { (void)cudaGetLastError(); return LST_ECUDA; }
  return bad(c, cudaGetLastError()) ? LST_ECUDA : LST_OK;
}

int lst_run_batch(lst_ctx* c, int32_t first, int32_t n, void* cuda_stream) {
  if (!c || first < 0 || n <= 0 || first + n > c->n_slots) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // The launch sequence has no per-run arguments, so it is captured once per (first, n) and replayed as a CUDA graph
  // (one submission instead of 19 launches + 2 memsets).  The legacy default stream cannot be captured: direct launches.
  if (c->use_graphs && st != nullptr && st != cudaStreamLegacy && st != cudaStreamPerThread) {
    const long long key = ((long long)first << 32) | (unsigned)n;
    auto it = c->graphs.find(key);
    if (it == c->graphs.end()) {
      cudaGraphExec_t exec = nullptr;
      if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        c->capturing = true;
        const int rc = run_sequence(c, first, n, st, nullptr);
        c->capturing = false;
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(st, &graph);
        if (rc == LST_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
        if (graph) cudaGraphDestroy(graph);
      }
      if (!exec) {                       // capture not possible here: stay with direct launches for this context
        (void)cudaGetLastError();
        c->use_graphs = false;
        c->sticky_cuda_error = false;
        return run_sequence(c, first, n, st, nullptr);
      }
      it = c->graphs.emplace(key, exec).first;
    }
    return bad(c, cudaGraphLaunch(it->second, st)) ? LST_ECUDA : LST_OK;
  }
  return run_sequence(c, first, n, st, nullptr);
}

int lst_run_batch_profile(lst_ctx* c, int32_t first, int32_t n, void* cuda_stream, float* h_ms) {
  if (!c || !h_ms || first < 0 || n <= 0 || first + n > c->n_slots) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaEvent_t ev[N_LAUNCHES + 2];
  for (auto& e : ev) if (bad(c, cudaEventCreate(&e))) return LST_ECUDA;
  int rc = run_sequence(c, first, n, st, ev);
  if (rc == LST_OK && bad(c, cudaStreamSynchronize(st))) rc = LST_ECUDA;
  if (rc == LST_OK)
    for (int i = 0; i <= N_LAUNCHES; ++i)
      if (bad(c, cudaEventElapsedTime(&h_ms[i], ev[i], ev[i + 1]))) { rc = LST_ECUDA; break; }
  for (auto& e : ev) cudaEventDestroy(e);
  return rc;
}

const char* lst_launch_name(int32_t i) {
  static const char* names[N_LAUNCHES + 1] = {
      "memset", "a0.hist", "a0.scan", "a0.scatter", "a0.rank", "a1.md_sweep", "a1.scan", "a1.md_finish", "a2.ls_sweep", "a2.scan", "a2.ls_finish",
      "a3.t3", "a4.t5", "a5.dnn", "a6.pls_bin", "a6.match5", "a6.pt5_lists", "a6.match3", "a6.tc_emit", "f1.tc_clean"};
  return (i >= 0 && i <= N_LAUNCHES) ? names[i] : nullptr;
}

int lst_run(lst_ctx* c, int32_t slot, void* cuda_stream) { return lst_run_batch(c, slot, 1, cuda_stream); }

int lst_get(lst_ctx* c, int32_t slot, int32_t objtype, lst_view* v) {
  if (!c || !v || slot < 0 || slot >= c->n_slots || objtype < 0 || objtype >= LST_N_OBJ) return LST_EINVAL;
  const Slot& s = c->h_slots[slot];
  *v = lst_view{};
  auto I = [](const void* p) { return static_cast<const int32_t*>(p); };
  switch (objtype) {
    case LST_OBJ_HIT: v->capacity = c->caps.max_hits; v->count = s.cnt + LST_CNT_HIT; v->i0 = s.hit_orig; v->i1 = s.sensor_start;
      v->f0 = reinterpret_cast<const float*>(s.hit); break;
    case LST_OBJ_MD: v->capacity = c->caps.max_md; v->count = s.cnt + LST_CNT_MD; v->i0 = I(s.md_hits); v->i1 = s.md_modt;
      v->i2 = s.md_start; v->f0 = reinterpret_cast<const float*>(s.md_pos); v->f1 = reinterpret_cast<const float*>(s.md_cw); break;
    case LST_OBJ_LS: v->capacity = c->caps.max_ls; v->count = s.cnt + LST_CNT_LS; v->i0 = I(s.ls_ab); v->i1 = s.ls_start; v->f0 = s.ls_c; break;
    case LST_OBJ_T3: v->capacity = c->caps.max_t3; v->count = s.cnt + LST_CNT_T3; v->i0 = I(s.t3_abc); v->i1 = s.t3_l1; v->i2 = s.t3_start;
      v->f0 = s.t3_k; break;
    case LST_OBJ_T5C: v->capacity = c->caps.max_t5c; v->count = s.cnt + LST_CNT_T5C; v->i0 = s.t5c_md; v->i1 = I(s.t5c_t3); v->i2 = s.t5c_pass;
      v->f0 = s.t5c_curv; v->f1 = s.t5c_feat; v->f2 = s.t5c_score; break;
    case LST_OBJ_T5: v->capacity = c->caps.max_t5; v->count = s.cnt + LST_CNT_T5; v->i0 = s.t5_list; break;
    case LST_OBJ_TC: v->capacity = c->caps.max_tc; v->count = s.cnt + LST_CNT_TC; v->i0 = s.tc; break;
    case LST_OBJ_MATCH5: v->capacity = c->caps.max_t5; v->count = s.cnt + LST_CNT_T5; v->i0 = s.best5; v->f0 = s.chi5; break;
    case LST_OBJ_GRAPH: v->capacity = c->caps.max_md; v->count = s.cnt + LST_CNT_MD; v->i0 = s.ls_start; v->i1 = s.g_col; v->i2 = I(s.md_hits);
      v->f0 = s.g_node; v->f1 = s.ls_c; break;
    case LST_OBJ_TCC: v->capacity = c->caps.max_tc; v->count = s.cnt + LST_CNT_TCC; v->i0 = s.tcc; break;
    case LST_OBJ_TCX: v->capacity = c->caps.max_tc; v->count = s.cnt + LST_CNT_TC; v->i0 = s.tc_keep; v->i1 = s.tc_hits; v->i2 = s.tc_q; break;
  }
  return LST_OK;
}

int lst_status(lst_ctx* c, int32_t slot, uint32_t* status_bits, int32_t* counts, void* cuda_stream) {
  if (!c || slot < 0 || slot >= c->n_slots) return LST_EINVAL;
  int32_t tmp[LST_N_CNT];
  if (bad(c, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)))) return LST_ECUDA;
  if (bad(c, cudaMemcpy(tmp, c->h_slots[slot].cnt, sizeof(tmp), cudaMemcpyDeviceToHost))) return LST_ECUDA;
  if (status_bits) *status_bits = static_cast<uint32_t>(tmp[LST_N_CNT - 1]);
  if (counts) for (int i = 0; i < LST_N_CNT; ++i) counts[i] = tmp[i];
  return LST_OK;
}

int lst_load_batch_host16(lst_ctx* c, int32_t first, int32_t n, const void* h_blob, size_t blob_bytes, void* cuda_stream) {
  if (!c || !h_blob || first < 0 || n <= 0 || first + n > c->n_slots) return LST_EINVAL;
  if (2 * (long long)c->n_modules > 65535) return LST_EINVAL;           // sensor keys must fit 16 bits
  if (c->sticky_cuda_error) return LST_ECUDA;
  const int32_t* desc = static_cast<const int32_t*>(h_blob);
  size_t need = blob_header_bytes(n);
  if (blob_bytes < need) return LST_EINVAL;
  for (int e = 0; e < n; ++e) {
    const int nh = desc[2 * e], np = desc[2 * e + 1];
    if (nh < 0 || np < 0 || nh > c->caps.max_hits || np > c->caps.max_pls) return LST_EINVAL;
    need += blob16_event_bytes(nh, np);
  }
  if (need > blob_bytes || need > c->batch_in_stride * n + 1024) return LST_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* dst = c->batch_in + c->batch_in_stride * first;
  if (bad(c, cudaMemcpyAsync(dst, h_blob, need, cudaMemcpyHostToDevice, st))) return LST_ECUDA;
  k_bind_batch16<<<(n + 63) / 64, 64, 0, st>>>(c->d_slots, first, n, dst);
  return bad(c, cudaGetLastError()) ? LST_ECUDA : LST_OK;
}

int lst_read_tc_host(lst_ctx* c, int32_t slot, int32_t* h_counts, int32_t* h_tc, int32_t max_rows, void* cuda_stream) {
  if (!c || slot < 0 || slot >= c->n_slots || !h_counts || max_rows < 0 || (max_rows > 0 && !h_tc)) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const Slot& s = c->h_slots[slot];
  if (max_rows > c->caps.max_tc) max_rows = c->caps.max_tc;
  if (max_rows > 0 && h_tc == h_counts + LST_N_CNT) {     // adjacent host buffers: counters (header copy) + rows in one copy
    if (bad(c, cudaMemcpyAsync(h_counts, s.tc_hdr, sizeof(int32_t) * (LST_N_CNT + 3 * (size_t)max_rows), cudaMemcpyDeviceToHost, st))) return LST_ECUDA;
    return LST_OK;
  }
  if (bad(c, cudaMemcpyAsync(h_counts, s.cnt, sizeof(int32_t) * LST_N_CNT, cudaMemcpyDeviceToHost, st))) return LST_ECUDA;
  if (max_rows > 0 && bad(c, cudaMemcpyAsync(h_tc, s.tc, sizeof(int32_t) * 3 * (size_t)max_rows, cudaMemcpyDeviceToHost, st)))
    return LST_ECUDA;
  return LST_OK;
}

int lst_load_batch_host(lst_ctx* c, int32_t first, int32_t n, const void* h_blob, size_t blob_bytes, void* cuda_stream) {
  if (!c || !h_blob || first < 0 || n <= 0 || first + n > c->n_slots) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  const int32_t* desc = static_cast<const int32_t*>(h_blob);
  size_t need = blob_header_bytes(n);
  if (blob_bytes < need) return LST_EINVAL;
  for (int e = 0; e < n; ++e) {
    const int nh = desc[2 * e], np = desc[2 * e + 1];
    if (nh < 0 || np < 0 || nh > c->caps.max_hits || np > c->caps.max_pls) return LST_EINVAL;
    need += blob_event_bytes(nh, np);
  }
  if (need > blob_bytes || need > c->batch_in_stride * n + 1024) return LST_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* dst = c->batch_in + c->batch_in_stride * first;
  if (bad(c, cudaMemcpyAsync(dst, h_blob, need, cudaMemcpyHostToDevice, st))) return LST_ECUDA;
  k_bind_batch<<<(n + 63) / 64, 64, 0, st>>>(c->d_slots, first, n, dst);
  return bad(c, cudaGetLastError()) ? LST_ECUDA : LST_OK;
}

static int read_tc_batch(lst_ctx* c, int32_t first, int32_t n, int32_t* h_out, int32_t max_rows, void* cuda_stream, bool hits) {
  if (!c || !h_out || first < 0 || n <= 0 || first + n > c->n_slots || max_rows < 0) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  if (max_rows > c->caps.max_tc) return LST_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int* dst = c->batch_out + c->batch_out_stride * first;
  if (hits) k_pack_tc<true><<<dim3(8, n), 256, 0, st>>>(c->d_slots + first, max_rows, dst);
  else k_pack_tc<false><<<dim3(8, n), 256, 0, st>>>(c->d_slots + first, max_rows, dst);
  if (bad(c, cudaGetLastError())) return LST_ECUDA;
  const size_t bytes = sizeof(int32_t) * (LST_N_CNT + (hits ? 13 : 3) * (size_t)max_rows) * n;
  return bad(c, cudaMemcpyAsync(h_out, dst, bytes, cudaMemcpyDeviceToHost, st)) ? LST_ECUDA : LST_OK;
}

int lst_read_tc_batch_host(lst_ctx* c, int32_t first, int32_t n, int32_t* h_out, int32_t max_rows, void* cuda_stream) {
  return read_tc_batch(c, first, n, h_out, max_rows, cuda_stream, false);
}

int lst_read_tc_hits_batch_host(lst_ctx* c, int32_t first, int32_t n, int32_t* h_out, int32_t max_rows, void* cuda_stream) {
  return read_tc_batch(c, first, n, h_out, max_rows, cuda_stream, true);
}

int lst_export_graph(lst_ctx* c, int32_t first, int32_t n, void* cuda_stream) {
  if (!c || first < 0 || n <= 0 || first + n > c->n_slots) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  int gx = (c->n_sm * 4 + n - 1) / n;
  if (gx < 4) gx = 4;
  k_graph_export<<<dim3(gx, n), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(c->d_slots + first);
  return bad(c, cudaGetLastError()) ? LST_ECUDA : LST_OK;
}

int lst_measure_fp32(lst_ctx* c, int32_t fused, float* h_tflops, void* cuda_stream) {
  if (!c || !h_tflops) return LST_EINVAL;
  if (c->sticky_cuda_error) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  float* scratch = reinterpret_cast<float*>(c->batch_out);
  // measurement only: a failure here is reported but does not disable the context (no sticky flag)
  cudaEvent_t a = nullptr, b = nullptr;
  if (cudaEventCreate(&a) != cudaSuccess) return LST_ECUDA;
  if (cudaEventCreate(&b) != cudaSuccess) { cudaEventDestroy(a); return LST_ECUDA; }
  const int blocks = c->n_sm * 8, iters = 8192;
  float best = 0.f;
  cudaError_t e = cudaSuccess;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {             // first repetition warms up
    e = cudaEventRecord(a, st);
    if (e != cudaSuccess) break;
    if (fused) k_fp32_probe<true><<<blocks, 256, 0, st>>>(scratch, iters);
    else k_fp32_probe<false><<<blocks, 256, 0, st>>>(scratch, iters);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventRecord(b, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    if (e != cudaSuccess) break;
    const double flop = 2.0 * 8.0 * iters * 256.0 * blocks;      // one multiply + one add per chain step, fused or not
    if (rep && ms > 0.f) best = fmaxf(best, (float)(flop / (ms * 1e-3) / 1e12));
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  if (e != cudaSuccess) return LST_ECUDA;
  *h_tflops = best;
  return LST_OK;
}

void lst_destroy(lst_ctx* c) {
  if (!c) return;
  for (auto& kv : c->graphs) cudaGraphExecDestroy(kv.second);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->side) cudaStreamDestroy(c->side);
  delete c;
}

}  // extern "C"
