// lst_pairs.cuh -- a1 (mini-doublets) and a2 (line segments): order-preserving row sweeps.
//
// Both stages test every cell of per-module rectangles (rows = inner objects of module m, columns = the
// module's candidate partners) and must emit the passing cells in the build order of SPEC.md 4.1-4.2
// (module, row, column).  A warp owns whole rows and walks their columns 32 at a time:
//   1. prefilter:  all 32 lanes evaluate the cheap conservative form of the cuts (lst_math.cuh) on 32 cells;
//                  survivors (a few %) are appended, in order, to a per-warp queue in shared memory;
//   2. exact:      whenever the queue holds >= 32 cells a full warp evaluates the exact SPEC.md arithmetic
//                  on them; a passing cell becomes a record (row, seq = its rank among the row's objects, payload);
//   3. place:      records go to an unordered per-slot buffer (one atomic per 32 records), the row's object
//                  count goes to the row table.  A multi-block look-back scan of the row table
//                  (k_scan_lb, lst_kernels.cuh) gives every row its first output position, and a scatter
//                  kernel writes record -> start[row] + seq.
// A row is never split between warps and a warp visits its rows and columns in ascending order, so `seq`
// depends only on the input (bit-reproducible output order), whatever the scheduling.
// a1: row = module (cells = lower x upper hits of the module, both contiguous in the sorted hit store); a warp packs the cells of
//     32 modules into one flat index space.
// a2: row = MD a; its columns are the MDs of the modules connected to module(a), which are a few contiguous MD ranges:
//     lst_create compresses every CSR row into runs of consecutive module ids (Geo::run_*), MDs are stored in module order, so
//     one run = one contiguous slice of md_pos / md_aux, and k_md_finish writes a per-module column table (end column and MD
//     offset of up to LS_TAB non-empty runs).  A warp takes a chunk of consecutive rows (launch-wide ticket), cuts it into
//     module segments and sweeps every segment columns-outer / rows-inner: 32 column MDs in registers against each row of the
//     segment (anchors in shared memory).  seq = the row's count so far (shared memory, per chunk) + rank within the batch.
// Capacity overflow (more objects than the record buffer holds): the scan flags it, and the DIRECT instantiation
// of the sweep runs the stage again (inside the finish kernel), writing start[row] + seq in place for positions below the
// capacity ("first cap objects in build order").
#pragma once
#include "lst_kernels.cuh"

namespace lst {

constexpr int PAIR_WARPS = 4;        // warps per block
constexpr int Q_CAP = 64;            // survivor queue / record staging per warp (drained / flushed at >= 32)
constexpr int RUN_CAP = 32;          // runs of a CSR row cached per warp at a time
constexpr int LS_ROWS = 16;          // consecutive MD rows a warp takes at a time: 16 in batched launches (measured 4 / 8 / 16 / 32 rows: 119 / 90 / 83 / 86 us),
                                     // 8 in launches of a few events, where more warps find work (single event: 27 vs 34 us)
constexpr int LS_TAB = 8;            // non-empty runs per module held by the precomputed column table
constexpr int MD_BIG = 1 << 20;      // modules with more cells than this are swept alone (64-bit sweep counter)

__device__ __forceinline__ unsigned lanemask_lt() { unsigned m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

__device__ __forceinline__ void divmod_small(int v, int d, int& q, int& r) {   // 0 <= v < 2^22, d > 0
  q = (int)(((float)v + 0.5f) * rcp_fast((float)d));
  r = v - q * d;
  if (r < 0) { --q; r += d; } else if (r >= d) { ++q; r -= d; }
}

// rank of every passing lane among the passing lanes with the same row, continued from the previous batch
// (carry = row and running count of the last object emitted so far).  Returns seq; updates the carry.
__device__ __forceinline__ int row_sequence(int row, bool pass, unsigned mask, unsigned lt, int lane, int& carry_row, int& carry_n,
                                            bool& last_of_row) {
  const unsigned peers = __match_any_sync(0xffffffffu, row) & mask;
  const int seq = __popc(peers & lt) + (row == carry_row ? carry_n : 0);
  last_of_row = pass && ((peers >> lane) >> 1) == 0u;
  if (mask) {
    const int hl = 31 - __clz(mask);
    carry_row = __shfl_sync(0xffffffffu, row, hl);
    carry_n = __shfl_sync(0xffffffffu, seq, hl) + 1;
  }
  return seq;
}

// ------------------------------------------------------------------------------------------------
// a1: row = module m; cells = (lower hit i, upper hit j), i-major
// ------------------------------------------------------------------------------------------------
struct MdWarp {   // per-warp shared memory
  int P[33]; int4 par[32]; float inv[32];     // non-empty modules of the warp's current group: first flat cell, (lb, ub, n_up, mtm), 1/n_up
  int q_lo[Q_CAP], q_up[Q_CAP], q_mt[Q_CAP];
  MdRec st[Q_CAP];
  const uint8_t* layer;                        // the modules' layers if the caller gave them (a6 surface ranges), else null
};

template <bool DIRECT>
__device__ __forceinline__ void md_emit(const Slot& s, const MdRec& r, int cap, const uint8_t* layer = nullptr) {      // final arrays of one MD
  const int pos = s.md_start[r.mtm >> 2] + r.seq;
  if (pos >= cap) return;
  const float4 h = s.hit[r.p_lo];
  const int mt = r.mtm & 3;
  s.md_hits[pos] = make_int2(s.hit_orig[r.p_lo], s.hit_orig[r.p_up]);
  s.md_modt[pos] = r.mtm;
  s.md_pos[pos] = h;                                  // anchor (x, y, z, r1)
  s.md_cw[pos] = make_float2(r.c, r.w);
  // (c, w and f with the prefilter margins folded in, 1/r): one load for the LS prefilter; the low two mantissa bits of f
  // carry the module type (they only widen the tolerance)
  const float fm_ = __int_as_float(__float_as_int(md_relf(mt) * 1.0001f) | mt);
  s.md_aux[pos] = make_float4(r.c, fmaf(r.w, 1.0001f, 3.0e-7f), fm_, 1.0f / h.w);
  if (DIRECT && layer && layer[r.mtm >> 2] != 255) {    // surface ranges for a6 (the record path aggregates them per block)
    const int sg = xs_surface(mt, layer[r.mtm >> 2], h.z);
    const unsigned ref = __float_as_uint((mt & 2) ? fabsf(h.z) : h.w);
    atomicMin(s.surf_lo + sg, ref); atomicMax(s.surf_hi + sg, ref); atomicMax(s.surf_rhi + sg, __float_as_uint(h.w));
  }
}

template <bool DIRECT>
__device__ __forceinline__ void md_flush(const Slot& s, MdWarp& W, int n, int lane, int cap) {
  if (DIRECT) {
    if (lane < n) md_emit<true>(s, W.st[lane], cap, W.layer);
    return;
  }
  int base = 0;
  if (lane == 0) base = atomicAdd(s.cnt + LST_CNT_FILL_MD, n);
  base = __shfl_sync(0xffffffffu, base, 0);
  if (lane < n && base + lane < cap) s.md_rec[base + lane] = W.st[lane];
}

// exact evaluation of the first `n` (<= 32) queued cells; passing ones become staged records; returns the new staging count
template <bool DIRECT>
__device__ __forceinline__ int md_drain(const Slot& s, MdWarp& W, int n, int sn, int lane, unsigned lt, int& carry_row, int& carry_n) {
  bool pass = false;
  int p_lo = 0, p_up = 0, mtm = -1 - lane;
  float c = 0.f, w = 0.f;
  if (lane < n) {
    p_lo = W.q_lo[lane]; p_up = W.q_up[lane]; mtm = W.q_mt[lane];
    const float4 h1 = s.hit[p_lo], h2 = s.hit[p_up];
    pass = md_eval(h1.x, h1.y, h1.z, h1.w, h2.x, h2.y, h2.z, h2.w, mtm & 3, c, w);
  }
  const unsigned mask = __ballot_sync(0xffffffffu, pass);
  bool last;
  const int seq = row_sequence(mtm, pass, mask, lt, lane, carry_row, carry_n, last);
  if (pass) {
    MdRec r; r.p_lo = p_lo; r.p_up = p_up; r.mtm = mtm; r.seq = seq; r.c = c; r.w = w; r.pad0 = 0; r.pad1 = 0;
    W.st[sn + __popc(mask & lt)] = r;
    if (!DIRECT && last) s.md_start[mtm >> 2] = seq + 1;        // objects of this module so far
  }
  return sn + __popc(mask);
}

// queue the prefilter survivors of one sweep (in lane order); a full warp of queued cells is evaluated at once and full
// warps of records are flushed
template <bool DIRECT>
__device__ __forceinline__ void md_push(const Slot& s, MdWarp& W, bool pre, int p_lo, int p_up, int mtm, int& qn, int& sn, int lane,
                                        unsigned lt, int& carry_row, int& carry_n, int cap) {
  const unsigned mask = __ballot_sync(0xffffffffu, pre);
  if (!mask) return;
  if (pre) { const int q = qn + __popc(mask & lt); W.q_lo[q] = p_lo; W.q_up[q] = p_up; W.q_mt[q] = mtm; }
  qn += __popc(mask);
  __syncwarp();
  if (qn < 32) return;
  sn = md_drain<DIRECT>(s, W, 32, sn, lane, lt, carry_row, carry_n);
  __syncwarp();
  const int rest = qn - 32;
  int a = 0, b = 0, c = 0;
  if (lane < rest) { a = W.q_lo[32 + lane]; b = W.q_up[32 + lane]; c = W.q_mt[32 + lane]; }
  __syncwarp();
  if (lane < rest) { W.q_lo[lane] = a; W.q_up[lane] = b; W.q_mt[lane] = c; }
  qn = rest;
  if (sn >= 32) {
    md_flush<DIRECT>(s, W, 32, lane, cap);
    __syncwarp();
    MdRec t{};
    if (lane < sn - 32) t = W.st[32 + lane];
    __syncwarp();
    if (lane < sn - 32) W.st[lane] = t;
    sn -= 32;
  }
  __syncwarp();
}

template <bool DIRECT>
__device__ __forceinline__ void md_sweep_body(const Slot& s, const Geo& geo, const Caps& caps, MdWarp* Wall) {
  const int lane = threadIdx.x & 31;
  MdWarp& W = Wall[threadIdx.x >> 5];
  const unsigned lt = lanemask_lt();
  const int M = geo.n_modules;
  const int* __restrict__ ss = s.sensor_start;
  const float4* __restrict__ hit = s.hit;
  const int cap = caps.max_md;
  const int n_warps = gridDim.x * PAIR_WARPS;
  int qn = 0, sn = 0, carry_row = -1, carry_n = 0;
  if (lane == 0) W.layer = geo.has_layer ? geo.xs_layer : nullptr;
  __syncwarp();
  // modules are interleaved over the warps (heavy inner-layer modules have consecutive ids).  A warp takes 32 of its modules
  // at a time (one round of range loads) and sweeps their cells as ONE flat index space, 32 cells per step: most modules
  // hold fewer than 32 cells, so per-module sweeps would leave most lanes idle.
  const int wid = blockIdx.x * PAIR_WARPS + (threadIdx.x >> 5);
  for (int mb = wid; mb < M; mb += n_warps * 32) {
    const int my_m = mb + lane * n_warps;
    int lb = 0, ub = 0, ue = 0, mt = 0;
    if (my_m < M) {
      lb = ss[2 * my_m]; ub = ss[2 * my_m + 1]; ue = ss[2 * my_m + 2]; mt = geo.modt[my_m];
      if (!DIRECT) s.md_start[my_m] = 0;
    }
    const int n_lo = ub - lb, n_up = ue - ub;
    const long long cells64 = (long long)n_lo * n_up;
    const bool big = cells64 > MD_BIG;
    const int cells = big ? 0 : (int)cells64;
    int inc = cells;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    const int total = __shfl_sync(0xffffffffu, inc, 31);
    const unsigned nz = __ballot_sync(0xffffffffu, cells > 0);
    __syncwarp();
    W.P[lane + 1] = total;                       // padding: the search never runs past the last non-empty module
    __syncwarp();
    if (cells > 0) {
      const int i = __popc(nz & lt);
      W.P[i] = inc - cells; W.par[i] = make_int4(lb, ub, n_up, (my_m << 2) | mt); W.inv[i] = rcp_fast((float)n_up);
    }
    __syncwarp();
    if (total > 0) {
      // lane's cell of sweep F: module k of the group (first sweep: binary search; later sweeps: k only moves forward), then
      // (i, j) inside the module.  The hits of the next sweep are loaded while the current one is tested.
      int k = 0;
      {
        const int f = min(lane, total - 1);
#pragma unroll
        for (int step = 16; step > 0; step >>= 1)
          if (W.P[k + step] <= f) k += step;
      }
      auto decode = [&](int F, int& p_lo, int& p_up, int& mtm) {
        const int f = min(F + lane, total - 1);
        while (W.P[k + 1] <= f) ++k;
        const int4 pr = W.par[k];
        const int loc = f - W.P[k];
        int i = (int)(((float)loc + 0.5f) * W.inv[k]);
        int j = loc - i * pr.z;
        if (j < 0) { --i; j += pr.z; } else if (j >= pr.z) { ++i; j -= pr.z; }
        p_lo = pr.x + i; p_up = pr.y + j; mtm = pr.w;
      };
      int n_lo_, n_up_, n_mt;
      decode(0, n_lo_, n_up_, n_mt);
      float4 n1 = __ldg(hit + n_lo_), n2 = __ldg(hit + n_up_);
      for (int F = 0; F < total; F += 32) {
        const int p_lo = n_lo_, p_up = n_up_, mtm = n_mt;
        const float4 h1 = n1, h2 = n2;
        if (F + 32 < total) { decode(F + 32, n_lo_, n_up_, n_mt); n1 = __ldg(hit + n_lo_); n2 = __ldg(hit + n_up_); }
        const bool pre = md_prefilter(h1.x, h1.y, h1.z, h1.w, h2.x, h2.y, h2.z, h2.w, mtm & 3) && (F + lane < total);
        md_push<DIRECT>(s, W, pre, p_lo, p_up, mtm, qn, sn, lane, lt, carry_row, carry_n, cap);
      }
    }
    // modules too large for the flat space (only in pathological events): alone, (i, j) advanced incrementally
    unsigned todo = __ballot_sync(0xffffffffu, big);
    while (todo) {
      const int kk = __ffs(todo) - 1;
      todo &= todo - 1;
      const int blb = __shfl_sync(0xffffffffu, lb, kk), bub = __shfl_sync(0xffffffffu, ub, kk), bue = __shfl_sync(0xffffffffu, ue, kk);
      const int mtm = ((mb + kk * n_warps) << 2) | __shfl_sync(0xffffffffu, mt, kk);
      const int bn_lo = bub - blb, bn_up = bue - bub;
      int i, j, q32, r32;                       // the lane's cell (i, j); 32 cells further = (+q32, +r32)
      divmod_small(lane, bn_up, i, j);
      divmod_small(32, bn_up, q32, r32);
      const long long n_sweeps = ((long long)bn_lo * bn_up + 31) >> 5;
      for (long long sw = 0; sw < n_sweeps; ++sw) {
        bool pre = false;
        const int p_lo = blb + i, p_up = bub + j;
        if (i < bn_lo) {
          const float4 h1 = __ldg(hit + p_lo), h2 = __ldg(hit + p_up);
          pre = md_prefilter(h1.x, h1.y, h1.z, h1.w, h2.x, h2.y, h2.z, h2.w, mtm & 3);
        }
        i += q32; j += r32;
        if (j >= bn_up) { j -= bn_up; ++i; }
        md_push<DIRECT>(s, W, pre, p_lo, p_up, mtm, qn, sn, lane, lt, carry_row, carry_n, cap);
      }
    }
  }
  if (qn) { sn = md_drain<DIRECT>(s, W, qn, sn, lane, lt, carry_row, carry_n); __syncwarp(); }
  if (sn >= 32) {
    md_flush<DIRECT>(s, W, 32, lane, cap);
    __syncwarp();
    MdRec t{};
    if (lane < sn - 32) t = W.st[32 + lane];
    __syncwarp();
    if (lane < sn - 32) W.st[lane] = t;
    sn -= 32;
    __syncwarp();
  }
  if (sn) md_flush<DIRECT>(s, W, sn, lane, cap);
}

#ifndef MD_MIN_BLOCKS
#define MD_MIN_BLOCKS 7
#endif
__global__ void __launch_bounds__(PAIR_WARPS * 32, MD_MIN_BLOCKS) k_md_sweep(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  pdl_begin();
  __shared__ MdWarp Wall[PAIR_WARPS];
  md_sweep_body<false>(slots[blockIdx.y], geo, caps, Wall);
}

__device__ __forceinline__ void ls_write_tables(const Slot& s, const Geo& geo);      // a2's per-module column tables (below)

// a1 finish (md_start holds the exclusive scan of the per-module counts by now): record -> md_start[module] + seq.
// If the stage overflowed its capacity the record buffer is incomplete: run the sweep again, writing in place.
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_md_finish(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  pdl_begin();
  __shared__ MdWarp Wall[PAIR_WARPS];
  const Slot& s = slots[blockIdx.y];
  if (s.cnt[CNT_STATUS] & LST_ST_OVF_MD) { ls_write_tables(s, geo); md_sweep_body<true>(s, geo, caps, Wall); return; }
  // One pass over max(records, modules): item j places record j and writes the LS column table of module j.  Both are
  // chains of dependent loads; all loads of a level are issued together (loads first, stores last), so an item costs
  // three memory round trips in all.
  const int n_rec = min(s.cnt[LST_CNT_FILL_MD], caps.max_md);
  const int M = geo.n_modules;
  const int* __restrict__ mds = s.md_start;
  // a6 surface ranges (reference coordinate of the anchors per barrel layer / disk side): per block in shared memory first
  __shared__ unsigned b_lo[XS_NS], b_hi[XS_NS], b_rh[XS_NS];
  if (threadIdx.x < XS_NS) { b_lo[threadIdx.x] = 0xFFFFFFFFu; b_hi[threadIdx.x] = 0u; b_rh[threadIdx.x] = 0u; }
  __syncthreads();
  LST_FOR_ITEMS(j, max(n_rec, M)) {
    const bool has_r = j < n_rec, has_m = j < M;
    // level 1
    MdRec r{};
    int e0 = 0, e1 = 0, m0 = 0, m1 = 0;
    if (has_r) r = s.md_rec[j];
    if (has_m) { e0 = __ldg(geo.run_ptr + j); e1 = __ldg(geo.run_ptr + j + 1); m0 = mds[j]; m1 = mds[j + 1]; }
    const bool tab_on = has_m && m1 > m0;               // modules without rows are never looked up
    // level 2
    int pos = 0, o_lo = 0, o_up = 0;
    float4 h = make_float4(0.f, 0.f, 0.f, 1.f);
    int lay = 0;
    if (has_r) {
      pos = mds[r.mtm >> 2] + r.seq; h = s.hit[r.p_lo]; o_lo = s.hit_orig[r.p_lo]; o_up = s.hit_orig[r.p_up];
      if (geo.has_layer) lay = geo.xs_layer[r.mtm >> 2];
    }
    int c0[LS_TAB], c1[LS_TAB], b0[LS_TAB], b1[LS_TAB];
#pragma unroll
    for (int q = 0; q < LS_TAB; ++q) { const bool in = tab_on && e0 + q < e1; c0[q] = in ? __ldg(geo.run_c0 + e0 + q) : 0; c1[q] = in ? __ldg(geo.run_c1 + e0 + q) : 0; }
    // level 3
#pragma unroll
    for (int q = 0; q < LS_TAB; ++q) { b0[q] = mds[c0[q]]; b1[q] = mds[c1[q]]; }
    // stores
    if (has_r && pos < caps.max_md) {
      const int mt = r.mtm & 3;
      s.md_hits[pos] = make_int2(o_lo, o_up);
      s.md_modt[pos] = r.mtm;
      s.md_pos[pos] = h;
      s.md_cw[pos] = make_float2(r.c, r.w);
      const float fm_ = __int_as_float(__float_as_int(md_relf(mt) * 1.0001f) | mt);
      s.md_aux[pos] = make_float4(r.c, fmaf(r.w, 1.0001f, 3.0e-7f), fm_, 1.0f / h.w);
      if (geo.has_layer && lay != 255) {
        const int sg = xs_surface(mt, lay, h.z);
        const unsigned ref = __float_as_uint((mt & 2) ? fabsf(h.z) : h.w);      // positive floats: bit order = value order
        atomicMin(&b_lo[sg], ref); atomicMax(&b_hi[sg], ref); atomicMax(&b_rh[sg], __float_as_uint(h.w));
      }
    }
    if (tab_on) {
      int ends[LS_TAB], dl[LS_TAB];
      int k = 0, L = 0;
#pragma unroll
      for (int q = 0; q < LS_TAB; ++q) {
        const int n = b1[q] - b0[q];
        if (n > 0) {
#pragma unroll
          for (int t = 0; t < LS_TAB; ++t) if (t == k) { dl[t] = b0[q] - L; ends[t] = L + n; }
          L += n; ++k;
        }
      }
      for (int e = e0 + LS_TAB; e < e1; ++e) {             // more than LS_TAB runs in the CSR row (rare)
        const int bb = mds[geo.run_c0[e]], n = mds[geo.run_c1[e]] - bb;
        if (n > 0) {
#pragma unroll
          for (int t = 0; t < LS_TAB; ++t) if (t == k) { dl[t] = bb - L; ends[t] = L + n; }
          L += n; ++k;
        }
      }
#pragma unroll
      for (int t = 0; t < LS_TAB; ++t) if (t >= k) { ends[t] = L; dl[t] = 0; }
      if (k > LS_TAB) ends[LS_TAB - 1] = -1;
      int4* tab = reinterpret_cast<int4*>(s.ls_tab + 2 * LS_TAB * (size_t)j);
      static_assert(LS_TAB == 8, "table layout");
      tab[0] = make_int4(ends[0], ends[1], ends[2], ends[3]); tab[1] = make_int4(ends[4], ends[5], ends[6], ends[7]);
      tab[2] = make_int4(dl[0], dl[1], dl[2], dl[3]); tab[3] = make_int4(dl[4], dl[5], dl[6], dl[7]);
    }
  }
  if (geo.has_layer) {
    __syncthreads();
    if (threadIdx.x < XS_NS && b_hi[threadIdx.x] != 0u) {
      atomicMin(s.surf_lo + threadIdx.x, b_lo[threadIdx.x]); atomicMax(s.surf_hi + threadIdx.x, b_hi[threadIdx.x]);
      atomicMax(s.surf_rhi + threadIdx.x, b_rh[threadIdx.x]);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a2: row = MD a of module m; columns = the MDs of the runs of CSR row m, ascending
// ------------------------------------------------------------------------------------------------
struct LsWarp {
  int r_off[RUN_CAP + 1], r_b0[RUN_CAP];      // non-empty runs of the current module: first column, (first MD) - (first column)
  float4 a_pos[LS_ROWS], a_aux[LS_ROWS];      // the rows of the current chunk: anchor, prefilter record (.w = -2 / r)
  __align__(16) int tab[LS_ROWS][2 * LS_TAB]; // ... and the column table of each row's module
  int cnt[LS_ROWS];                           // LSs found so far in each row of the chunk
  int rmask;                                  // rows per chunk - 1
  int q_a[Q_CAP], q_b[Q_CAP];
  LsRec st[Q_CAP];
};

__device__ __forceinline__ Anchor load_anchor(const Slot& s, int i) {
  const float4 p = s.md_pos[i];
  const float2 q = s.md_cw[i];
  Anchor a; a.x = p.x; a.y = p.y; a.z = p.z; a.r = p.w; a.c = q.x; a.w = q.y; a.mt = s.md_modt[i] & 3;
  return a;
}

template <bool DIRECT>
__device__ __forceinline__ void ls_flush(const Slot& s, LsWarp& W, int n, int lane, int cap) {
  if (DIRECT) {
    if (lane < n) {
      const LsRec r = W.st[lane];
      const int pos = s.ls_start[r.a] + r.seq;
      if (pos < cap) { s.ls_ab[pos] = make_int2(r.a, r.b); s.ls_c[pos] = r.c; }
    }
    return;
  }
  int base = 0;
  if (lane == 0) base = atomicAdd(s.cnt + LST_CNT_FILL_LS, n);
  base = __shfl_sync(0xffffffffu, base, 0);
  if (lane < n && base + lane < cap) s.ls_rec[base + lane] = W.st[lane];
}

// exact evaluation of the first `n` (<= 32) queued cells.  The queue holds cells of the current chunk only, and the cells of
// one row arrive in ascending column order, so seq = (LSs of the row so far) + (rank among the row's passing cells of this batch).
template <bool DIRECT>
__device__ __forceinline__ int ls_drain(const Slot& s, LsWarp& W, int n, int sn, int lane, unsigned lt) {
  bool pass = false;
  int a = -1 - lane, b = 0;
  float c = 0.f;
  if (lane < n) {
    a = W.q_a[lane]; b = W.q_b[lane];
    const Anchor A = load_anchor(s, a), B = load_anchor(s, b);
    pass = ls_eval(A, B, c);
  }
  const unsigned mask = __ballot_sync(0xffffffffu, pass);
  if (!mask) return sn;
  const unsigned peers = __match_any_sync(0xffffffffu, a) & mask;
  if (pass) {
    const int before = __popc(peers & lt);
    LsRec r; r.a = a; r.b = b; r.seq = W.cnt[a & W.rmask] + before; r.c = c;
    W.st[sn + __popc(mask & lt)] = r;
  }
  __syncwarp();
  if (pass && (peers >> lane) >> 1 == 0u) W.cnt[a & W.rmask] += __popc(peers);      // last passing cell of its row in this batch
  return sn + __popc(mask);
}

template <bool DIRECT>
__device__ __forceinline__ void ls_flush_full(const Slot& s, LsWarp& W, int& sn, int lane, int cap) {
  if (sn < 32) return;
  __syncwarp();
  ls_flush<DIRECT>(s, W, 32, lane, cap);
  __syncwarp();
  LsRec tr{};
  if (lane < sn - 32) tr = W.st[32 + lane];
  __syncwarp();
  if (lane < sn - 32) W.st[lane] = tr;
  sn -= 32;
  __syncwarp();
}

// non-empty runs [e, e + 32) of CSR row m -> the warp's run table; returns the number of columns they hold
__device__ __forceinline__ int ls_load_runs(const Geo& geo, const int* __restrict__ mds, LsWarp& W, int e0, int e1, int lane, unsigned lt) {
  const int e = e0 + lane;
  int b0 = 0, n = 0;
  if (e < e1) { b0 = mds[geo.run_c0[e]]; n = mds[geo.run_c1[e]] - b0; }
  int inc = n;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
  const unsigned nz = __ballot_sync(0xffffffffu, n > 0);
  const int total = __shfl_sync(0xffffffffu, inc, 31);
  __syncwarp();
  W.r_off[lane + 1] = total;                    // padding for the search
  __syncwarp();
  if (n > 0) { const int i = __popc(nz & lt); W.r_off[i] = inc - n; W.r_b0[i] = b0 - (inc - n); }
  __syncwarp();
  return total;
}
// column t of the run table -> MD index
__device__ __forceinline__ int ls_column(const LsWarp& W, int t) {
  int r = 0;
#pragma unroll
  for (int step = RUN_CAP / 2; step > 0; step >>= 1)
    if (W.r_off[r + step] <= t) r += step;
  return W.r_b0[r] + t;
}

// per-module column table for the LS sweep: [0, LS_TAB) = last column + 1 of each non-empty run (padded with the module's
// column count L, so entry LS_TAB - 1 is L), [LS_TAB, 2 LS_TAB) = (first MD) - (first column) of each run.  More than LS_TAB
// non-empty runs: entry LS_TAB - 1 = -1 and the sweep builds its run table itself.
__device__ __forceinline__ void ls_write_tables(const Slot& s, const Geo& geo) {
  const int* __restrict__ mds = s.md_start;
  LST_FOR_ITEMS(m, geo.n_modules) {
    int* tab = s.ls_tab + 2 * LS_TAB * (size_t)m;
    if (mds[m] == mds[m + 1]) continue;                 // no rows: never read
    int k = 0, L = 0;
    for (int e = geo.run_ptr[m], e1 = geo.run_ptr[m + 1]; e < e1; e += 8) {      // 8 runs at a time: their loads are independent
      int c0[8], c1[8], b0[8], b1[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) { const bool in = e + j < e1; c0[j] = in ? __ldg(geo.run_c0 + e + j) : 0; c1[j] = in ? __ldg(geo.run_c1 + e + j) : 0; }
#pragma unroll
      for (int j = 0; j < 8; ++j) { b0[j] = mds[c0[j]]; b1[j] = mds[c1[j]]; }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int n = b1[j] - b0[j];
        if (n > 0) {
          if (k < LS_TAB) { tab[LS_TAB + k] = b0[j] - L; tab[k] = L + n; }
          L += n; ++k;
        }
      }
    }
    for (int j = k; j < LS_TAB; ++j) { tab[j] = L; tab[LS_TAB + j] = 0; }
    if (k > LS_TAB) tab[LS_TAB - 1] = -1;
  }
}

template <bool DIRECT>
__device__ __forceinline__ void ls_push(const Slot& s, LsWarp& W, bool pre, int a, int b, int& qn, int& sn, int lane, unsigned lt, int cap) {
  const unsigned mask = __ballot_sync(0xffffffffu, pre);
  if (!mask) return;
  if (pre) { const int q = qn + __popc(mask & lt); W.q_a[q] = a; W.q_b[q] = b; }
  qn += __popc(mask);
  if (qn < 32) return;
  __syncwarp();
  sn = ls_drain<DIRECT>(s, W, 32, sn, lane, lt);
  __syncwarp();
  const int rest = qn - 32;
  int x = 0, y = 0;
  if (lane < rest) { x = W.q_a[32 + lane]; y = W.q_b[32 + lane]; }
  __syncwarp();
  if (lane < rest) { W.q_a[lane] = x; W.q_b[lane] = y; }
  qn = rest;
  ls_flush_full<DIRECT>(s, W, sn, lane, cap);
  __syncwarp();
}

// A warp takes LS_ROWS consecutive MDs (rows) at a time.  Rows of the same module share their columns, so the chunk is cut
// into module segments and every segment is swept columns-outer / rows-inner: the 32 column MDs of a step are loaded once
// into registers (next step's loads already in flight) and tested against each row of the segment, whose anchors sit in
// shared memory (broadcast reads).  The survivor queue is emptied at the end of every chunk, so the per-row LS counts live in
// shared memory for the duration of a chunk and the row table is written once, coalesced.
// one step: the 32 column MDs (bc, Bpc, Bac) against rows [i0, i1) of the chunk
template <bool DIRECT>
__device__ __forceinline__ void ls_rows(const Slot& s, LsWarp& W, int a0, int i0, int i1, bool valid, int bc, float4 Bpc, float4 Bac, int& qn, int& sn,
                                        int lane, unsigned lt, int cap) {
  int i = i0;
  for (; i + 1 < i1; i += 2) {             // two rows in flight: independent prefilter chains
    const float4 Ap0 = W.a_pos[i], Aa0 = W.a_aux[i], Ap1 = W.a_pos[i + 1], Aa1 = W.a_aux[i + 1];
    const bool pre0 = ls_prefilter(Ap0, Aa0, Aa0.w, Bpc, Bac) && valid;
    const bool pre1 = ls_prefilter(Ap1, Aa1, Aa1.w, Bpc, Bac) && valid;
    ls_push<DIRECT>(s, W, pre0, a0 + i, bc, qn, sn, lane, lt, cap);
    ls_push<DIRECT>(s, W, pre1, a0 + i + 1, bc, qn, sn, lane, lt, cap);
  }
  if (i < i1) {
    const float4 Ap0 = W.a_pos[i], Aa0 = W.a_aux[i];
    const bool pre0 = ls_prefilter(Ap0, Aa0, Aa0.w, Bpc, Bac) && valid;
    ls_push<DIRECT>(s, W, pre0, a0 + i, bc, qn, sn, lane, lt, cap);
  }
}

// slow path (module with more than LS_TAB non-empty runs): run table built here, one column step after the other
template <bool DIRECT>
__device__ __forceinline__ void ls_sweep_columns(const Slot& s, LsWarp& W, int L, int a0, int i0, int i1, int& qn, int& sn, int lane, unsigned lt, int cap) {
  for (int t0 = 0; t0 < L; t0 += 32) {
    const int b = ls_column(W, min(t0 + lane, L - 1));
    ls_rows<DIRECT>(s, W, a0, i0, i1, t0 + lane < L, b, __ldg(s.md_pos + b), __ldg(s.md_aux + b), qn, sn, lane, lt, cap);
  }
}

// column t of a module's column table (k_md_finish) -> MD index
__device__ __forceinline__ int ls_tab_column(const int* tab, int t) {
  int r = (tab[3] <= t) ? 4 : 0;
  if (tab[r + 1] <= t) r += 2;
  if (tab[r] <= t) r += 1;                    // r = number of runs that end at or before t (entry LS_TAB - 1 = L > t)
  return t + tab[LS_TAB + r];
}

// The chunks (`rows` consecutive MDs, 8 or 16) of ALL the events of a launch are handed out by one atomic ticket (kept in the
// first slot; the next ticket is fetched while the current chunk is swept), so every warp of the persistent grid works until
// the whole launch is done.  Rows of the same module share their columns, so a chunk is cut into module segments and every
// segment is swept columns-outer / rows-inner: the 32 column MDs of a step are loaded once into registers and tested against
// each row of the segment, whose anchors sit in shared memory (broadcast reads).  The (segment, step) pairs of a chunk form
// one sequence and the column loads of the next pair -- possibly of the next segment -- are in flight while the current one
// is tested; the column tables of all the chunk's modules are fetched together at the start of the chunk, so a chunk costs
// three dependent memory round trips (rows, tables, first columns) however many modules it spans.  The survivor queue is
// emptied at the end of every chunk, so the per-row LS counts live in shared memory for the duration of a chunk and the
// row table is written once, coalesced.  Which warp sweeps which chunk does not matter: a record carries its row and its
// rank in the row.
template <bool DIRECT>
__device__ __forceinline__ void ls_sweep_body(const Slot* __restrict__ slots, int n_ev, int rows, const Geo& geo, const Caps& caps, LsWarp* Wall) {
  const int lane = threadIdx.x & 31;
  LsWarp& W = Wall[threadIdx.x >> 5];
  const unsigned lt = lanemask_lt();
  const int cap = caps.max_ls;
  // chunks of events [0, lane] (inclusive scan over the events of the launch; at most 32 events per ticket)
  int cum = 0;
  if (lane == 0) W.rmask = rows - 1;
  if (lane < n_ev) cum = (slots[lane].cnt[LST_CNT_MD] + rows - 1) / rows;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, cum, d); if (lane >= d) cum += t; }
  int* ticket = slots[0].tk + (DIRECT ? TK_LS_DIRECT : TK_LS_SWEEP);
  int qn = 0, sn = 0;
  int next = 0;
  if (lane == 0) next = atomicAdd(ticket, 1);
  int ev_prev = -1;
  while (true) {
    const int T = __shfl_sync(0xffffffffu, next, 0);
    const int ev = __popc(__ballot_sync(0xffffffffu, lane < n_ev && cum <= T));
    if (ev >= n_ev) break;
    if (lane == 0) next = atomicAdd(ticket, 1);
    const int first = __shfl_sync(0xffffffffu, cum, max(ev - 1, 0));
    const int a0 = (T - (ev ? first : 0)) * rows;
    if (ev != ev_prev && sn) { __syncwarp(); ls_flush<DIRECT>(slots[ev_prev], W, sn, lane, cap); sn = 0; __syncwarp(); }      // records go to their own event
    ev_prev = ev;
    const Slot& s = slots[ev];
    const float4* __restrict__ mpos = s.md_pos;
    const float4* __restrict__ maux = s.md_aux;
    const int n_rows = min(rows, s.cnt[LST_CNT_MD] - a0);
    int my_m = -1;
    __syncwarp();
    if (lane < n_rows) {
      const float4 aux = __ldg(maux + a0 + lane);
      W.a_pos[lane] = __ldg(mpos + a0 + lane); W.a_aux[lane] = make_float4(aux.x, aux.y, aux.z, -2.0f * aux.w);      // .w = -2 / r
      my_m = s.md_modt[a0 + lane] >> 2;
    }
    if (lane < LS_ROWS) W.cnt[lane] = 0;
    {
      static_assert(LS_TAB == 8, "four int4 per table");
#pragma unroll
      for (int r0 = 0; r0 < LS_ROWS; r0 += 8) if (r0 < rows) {           // one int4 of the tables per lane and round
        const int row = r0 + (lane >> 2), m_r = __shfl_sync(0xffffffffu, my_m, row);
        if (m_r >= 0) reinterpret_cast<int4*>(W.tab[row])[lane & 3] = __ldg(reinterpret_cast<const int4*>(s.ls_tab + 2 * LS_TAB * (size_t)m_r) + (lane & 3));
      }
    }
    const int prev_m = __shfl_up_sync(0xffffffffu, my_m, 1);
    const unsigned segs = __ballot_sync(0xffffffffu, lane < n_rows && (lane == 0 || my_m != prev_m));    // first rows of the module segments
    __syncwarp();
    unsigned todo = segs, slow = 0;
    int ni0 = 0, ni1 = 0, nL = 0, nt0 = 0;
    auto pop = [&]() -> bool {                // next segment with columns; segments that need the slow path are set aside
      while (todo) {
        ni0 = __ffs(todo) - 1; todo &= todo - 1;
        ni1 = todo ? __ffs(todo) - 1 : n_rows;
        nL = W.tab[ni0][LS_TAB - 1];
        if (nL > 0) return true;
        if (nL < 0) slow |= 1u << ni0;
      }
      return false;
    };
    bool have = pop();
    int b = 0;
    float4 Bp = make_float4(0.f, 0.f, 0.f, 1.f), Ba = Bp;
    if (have) { b = ls_tab_column(W.tab[ni0], min(lane, nL - 1)); Bp = __ldg(mpos + b); Ba = __ldg(maux + b); }
    while (have) {
      const int i0 = ni0, i1 = ni1, bc = b;
      const float4 Bpc = Bp, Bac = Ba;
      const bool valid = nt0 + lane < nL;
      if (nt0 + 32 < nL) nt0 += 32; else { have = pop(); nt0 = 0; }
      if (have) { b = ls_tab_column(W.tab[ni0], min(nt0 + lane, nL - 1)); Bp = __ldg(mpos + b); Ba = __ldg(maux + b); }      // next pair, ahead of use
      ls_rows<DIRECT>(s, W, a0, i0, i1, valid, bc, Bpc, Bac, qn, sn, lane, lt, cap);
    }
    while (slow) {                            // modules with more than LS_TAB non-empty runs
      const int i0 = __ffs(slow) - 1;
      slow &= slow - 1;
      const unsigned rest = segs & ~((2u << i0) - 1u);
      const int i1 = rest ? __ffs(rest) - 1 : n_rows;
      const int m = __shfl_sync(0xffffffffu, my_m, i0);
      const int e0 = geo.run_ptr[m], e1 = geo.run_ptr[m + 1];
      for (int eb = e0; eb < e1; eb += RUN_CAP) {                // one pass unless the CSR row has more than RUN_CAP runs
        const int L2 = ls_load_runs(geo, s.md_start, W, eb, min(eb + RUN_CAP, e1), lane, lt);
        if (L2 > 0) ls_sweep_columns<DIRECT>(s, W, L2, a0, i0, i1, qn, sn, lane, lt, cap);
      }
    }
    // end of the chunk: empty the queue, then the chunk's row counts are final
    if (qn) { __syncwarp(); sn = ls_drain<DIRECT>(s, W, qn, sn, lane, lt); qn = 0; ls_flush_full<DIRECT>(s, W, sn, lane, cap); }
    __syncwarp();
    if (!DIRECT && lane < n_rows) s.ls_start[a0 + lane] = W.cnt[lane];
  }
  __syncwarp();
  if (sn) ls_flush<DIRECT>(slots[ev_prev], W, sn, lane, cap);
}

// grid (persistent blocks, groups of up to 32 events)
#ifndef LS_MIN_BLOCKS
#define LS_MIN_BLOCKS 7            // 72 registers: 28 warps per SM measured best (64 / 56 registers spill, 84 leave 20 warps)
#endif
__global__ void __launch_bounds__(PAIR_WARPS * 32, LS_MIN_BLOCKS) k_ls_sweep(const Slot* __restrict__ slots, int n_ev, Geo geo, Caps caps) {
  pdl_begin();
  __shared__ LsWarp Wall[PAIR_WARPS];
  ls_sweep_body<false>(slots + 32 * blockIdx.y, min(32, n_ev - 32 * (int)blockIdx.y), n_ev < 8 ? 8 : LS_ROWS, geo, caps, Wall);
}

// a2 finish (ls_start holds the exclusive scan of the per-row counts by now): record -> ls_start[a] + seq; on capacity
// overflow the sweep runs again, in place
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_ls_finish(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  pdl_begin();
  __shared__ LsWarp Wall[PAIR_WARPS];
  const Slot& s = slots[blockIdx.y];
  if (s.cnt[CNT_STATUS] & LST_ST_OVF_LS) { ls_sweep_body<true>(slots + blockIdx.y, 1, 8, geo, caps, Wall); return; }
  const int n_rec = min(s.cnt[LST_CNT_FILL_LS], caps.max_ls);
  LST_FOR_ITEMS(j, n_rec) {
    const LsRec r = s.ls_rec[j];
    const int pos = s.ls_start[r.a] + r.seq;
    s.ls_ab[pos] = make_int2(r.a, r.b);
    s.ls_c[pos] = r.c;
  }
}

}  // namespace lst
