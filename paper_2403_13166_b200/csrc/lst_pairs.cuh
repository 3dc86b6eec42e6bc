// lst_pairs.cuh -- pair-parallel MD (a1) and LS (a2) kernels.
//
// Both stages test every cell of a per-module rectangle: rows = inner objects of module m (lower hits /
// MDs of m), columns = the module's candidate partners (upper hits of m / MDs of the CSR-connected
// modules), and the build order of SPEC.md 4.1-4.2 is row-major inside the module.  A warp sweeps the
// rectangle 32 cells at a time (narrow rectangles pack several rows into one sweep), so all 32 lanes
// evaluate a cut at once instead of one thread looping over its own row.
//
// Single evaluation, deterministic order:
//   1. pairs:    every passing pair becomes a record (row, rank inside the row, payload) appended to an
//                unordered per-slot record buffer (warp-staged in shared memory, one atomicAdd per flush);
//                the row's pass count goes to the scan array (md_off / ls_start).
//   2. scan:     exclusive scan of the row counts (k_scan), clamped to capacity, overflow flagged.
//   3. finalize: one thread per record scatters it to scan[row] + rank -- the SPEC.md build order.
// When a stage overflows its capacity the record buffer (same capacity) has dropped arbitrary records;
// the thread-per-row fill kernels of lst_kernels.cuh then rewrite the first `cap` objects in build
// order (they return immediately unless the stage's overflow bit is set).
#pragma once
#include "lst_kernels.cuh"

namespace lst {

constexpr int PAIR_WARPS = 8;        // warps per block
constexpr int STAGE_CAP = 64;        // staged records per warp (flush at >= 32)
constexpr int ITEMS_PER_WARP = 4;    // consecutive work items a warp takes at a time
constexpr int CAND_CAP = 512;        // candidate-MD index table per warp (shared memory)

__device__ __forceinline__ unsigned lanemask_lt() { unsigned m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

template <typename Rec>
__device__ __forceinline__ void flush_stage(Rec* __restrict__ stage, int& staged, int* counter, Rec* __restrict__ out, int cap, int lane) {
  int base = 0;
  if (lane == 0) base = atomicAdd(counter, staged);
  base = __shfl_sync(0xffffffffu, base, 0);
  for (int i = lane; i < staged; i += 32)
    if (base + i < cap) out[base + i] = stage[i];
  staged = 0;
  __syncwarp();
}

// largest m in [0, M) with off[m] <= i (off non-decreasing, off[0] = 0 <= i < off[M]): 32-ary search, the
// warp probes 32 positions per round
__device__ __forceinline__ int find_module(const int* __restrict__ off, int M, int i, int lane) {
  int lo = 0, n = M;
  while (n > 1) {
    const int step = (n + 31) >> 5;
    const int idx = lo + lane * step;
    const bool le = (idx < lo + n) && (off[idx] <= i);
    const int j = __popc(__ballot_sync(0xffffffffu, le)) - 1;
    const int nlo = lo + j * step;
    n = min(step, lo + n - nlo);
    lo = nlo;
  }
  return lo;
}

// ------------------------------------------------------------------------------------------------
// a1 pairs: rows = lower hits of m, columns = upper hits of m
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_md_pairs(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  __shared__ MdRec stage_all[PAIR_WARPS][STAGE_CAP];
  const Slot& s = slots[blockIdx.y];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  MdRec* stage = stage_all[warp];
  const unsigned lt = lanemask_lt();
  int staged = 0;
  const int M = geo.n_modules;
  const int* __restrict__ ioff = s.md_item_off;
  const int* __restrict__ ss = s.sensor_start;
  const float4* __restrict__ hit = s.hit;
  const int T = ioff[M];
  const int n_chunks = (T + ITEMS_PER_WARP - 1) / ITEMS_PER_WARP;
  for (int chunk = blockIdx.x * PAIR_WARPS + warp; chunk < n_chunks; chunk += gridDim.x * PAIR_WARPS) {
    const int i_end = min(T, (chunk + 1) * ITEMS_PER_WARP);
    int m_end = -1, m_beg = 0, m = 0;
    int lb = 0, ub = 0, n_lo = 0, L = 0, mt = 0;
    ItemPlan pl{};
    for (int i = chunk * ITEMS_PER_WARP; i < i_end; ++i) {
      if (i >= m_end) {   // next module
        m = find_module(ioff, M, i, lane);
        m_beg = ioff[m]; m_end = ioff[m + 1];
        lb = ss[2 * m]; ub = ss[2 * m + 1];
        n_lo = ub - lb; L = ss[2 * m + 2] - ub;
        mt = geo.modt[m];
        pl = item_plan(n_lo, L);
      }
      const int row0 = (i - m_beg) * pl.rows_per_item;
      const int row1 = min(n_lo, row0 + pl.rows_per_item);
      if (pl.S == 1) {
        // narrow rectangle: W columns per row, R = 32/W rows per sweep; the lane's column is fixed
        const int W = pl.W, lw = lane & (W - 1), rs = lane / W;
        const bool vcol = lw < L;
        const int pj = ub + min(lw, L - 1);
        const float4 h2 = hit[pj];
        const unsigned rowmask = (W == 32) ? 0xffffffffu : (((1u << W) - 1u) << (rs * W));
        for (int r0 = row0; r0 < row1; r0 += pl.R) {
          const int row = r0 + rs;
          const int pi = lb + min(row, n_lo - 1);
          const float4 h1 = hit[pi];
          const float r1 = fq(fa(fm(h1.x, h1.x), fm(h1.y, h1.y)));
          float c = 0.f, w = 0.f;
          const bool pass = vcol && row < row1 && md_eval(h1.x, h1.y, h1.z, r1, h2.x, h2.y, h2.z, mt, c, w);
          const unsigned mask = __ballot_sync(0xffffffffu, pass);
          if (mask) {
            const unsigned rm = mask & rowmask;
            if (lw == 0 && row < row1 && rm) s.md_off[pi] = __popc(rm);
            if (pass) {
              MdRec rec; rec.p_lo = pi; rec.p_up = pj; rec.rank = __popc(rm & lt); rec.modt = (m << 2) | mt;
              rec.c = c; rec.w = w; rec.r1 = r1; rec.pad = 0.f;
              stage[staged + __popc(mask & lt)] = rec;
            }
            staged += __popc(mask);
            __syncwarp();
            if (staged >= 32) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_MD, s.md_rec, caps.max_md, lane);
          }
        }
      } else {
        // wide rectangle: one row at a time, S sweeps per row
        for (int row = row0; row < row1; ++row) {
          const int pi = lb + row;
          const float4 h1 = hit[pi];
          const float r1 = fq(fa(fm(h1.x, h1.x), fm(h1.y, h1.y)));
          int running = 0;
          for (int sw = 0; sw < pl.S; ++sw) {
            const int col = sw * 32 + lane;
            const int pj = ub + min(col, L - 1);
            const float4 h2 = hit[pj];
            float c = 0.f, w = 0.f;
            const bool pass = col < L && md_eval(h1.x, h1.y, h1.z, r1, h2.x, h2.y, h2.z, mt, c, w);
            const unsigned mask = __ballot_sync(0xffffffffu, pass);
            if (mask) {
              if (pass) {
                MdRec rec; rec.p_lo = pi; rec.p_up = pj; rec.rank = running + __popc(mask & lt); rec.modt = (m << 2) | mt;
                rec.c = c; rec.w = w; rec.r1 = r1; rec.pad = 0.f;
                stage[staged + __popc(mask & lt)] = rec;
              }
              staged += __popc(mask);
              running += __popc(mask);
              __syncwarp();
              if (staged >= 32) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_MD, s.md_rec, caps.max_md, lane);
            }
          }
          if (lane == 0 && running) s.md_off[pi] = running;
        }
      }
    }
  }
  if (staged) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_MD, s.md_rec, caps.max_md, lane);
}

// a1 finalize: scatter the records to build order; candidate count L of every module for the LS sweep
__global__ void __launch_bounds__(256) k_md_final(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  const Slot& s = slots[blockIdx.y];
  const int n_rec = min(s.cnt[LST_CNT_TMP_MD], caps.max_md);
  LST_FOR_ITEMS(i, n_rec) {
    const MdRec rec = s.md_rec[i];
    const int pos = s.md_off[rec.p_lo] + rec.rank;
    if (pos < caps.max_md) {
      const float4 h1 = s.hit[rec.p_lo];
      s.md_hits[pos] = make_int2(s.hit_orig[rec.p_lo], s.hit_orig[rec.p_up]);
      s.md_modt[pos] = rec.modt;
      s.md_pos[pos] = make_float4(h1.x, h1.y, h1.z, rec.r1);
      s.md_cw[pos] = make_float2(rec.c, rec.w);
    }
  }
  LST_FOR_ITEMS(m, geo.n_modules) {
    int L = 0;
    const int e1 = geo.rowptr[m + 1];
    if (s.md_start[m + 1] > s.md_start[m])
      for (int e = geo.rowptr[m]; e < e1; ++e) { const int m2 = geo.col[e]; L += s.md_start[m2 + 1] - s.md_start[m2]; }
    s.ls_L[m] = L;
    s.ls_item_off[m] = item_plan(s.md_start[m + 1] - s.md_start[m], L).n_items;
  }
}

// ------------------------------------------------------------------------------------------------
// a2 pairs: rows = MDs of m, columns = MDs of the CSR-connected modules (ascending MD index)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ Anchor load_anchor2(const float4* __restrict__ pos, const float2* __restrict__ cw,
                                               const int* __restrict__ modt, int i) {
  const float4 p = pos[i];
  const float2 q = cw[i];
  Anchor a; a.x = p.x; a.y = p.y; a.z = p.z; a.r = p.w; a.c = q.x; a.w = q.y; a.mt = modt[i] & 3;
  return a;
}

// column -> MD index by walking the CSR row (only for rows with more than CAND_CAP candidates)
__device__ __noinline__ int cand_walk(const Slot& s, const Geo& geo, int m, int col) {
  const int e1 = geo.rowptr[m + 1];
  for (int e = geo.rowptr[m]; e < e1; ++e) {
    const int m2 = geo.col[e];
    const int b0 = s.md_start[m2], n = s.md_start[m2 + 1] - b0;
    if (col < n) return b0 + col;
    col -= n;
  }
  return 0;
}

__global__ void __launch_bounds__(PAIR_WARPS * 32) k_ls_pairs(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  __shared__ LsRec stage_all[PAIR_WARPS][STAGE_CAP];
  __shared__ int cand_all[PAIR_WARPS][CAND_CAP];
  const Slot& s = slots[blockIdx.y];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  LsRec* stage = stage_all[warp];
  int* cand = cand_all[warp];
  const unsigned lt = lanemask_lt();
  int staged = 0;
  const int M = geo.n_modules;
  const int* __restrict__ ioff = s.ls_item_off;
  const int* __restrict__ mds = s.md_start;
  const float4* __restrict__ mpos = s.md_pos;
  const float2* __restrict__ mcw = s.md_cw;
  const int* __restrict__ mmodt = s.md_modt;
  const int T = ioff[M];
  const int n_chunks = (T + ITEMS_PER_WARP - 1) / ITEMS_PER_WARP;
  for (int chunk = blockIdx.x * PAIR_WARPS + warp; chunk < n_chunks; chunk += gridDim.x * PAIR_WARPS) {
    const int i_end = min(T, (chunk + 1) * ITEMS_PER_WARP);
    int m_end = -1, m_beg = 0, m = 0, a0 = 0, n_m = 0, L = 0;
    bool tabled = false;
    ItemPlan pl{};
    for (int i = chunk * ITEMS_PER_WARP; i < i_end; ++i) {
      if (i >= m_end) {   // next module: candidate table cand[col] = MD index over the connected modules' MD ranges
        m = find_module(ioff, M, i, lane);
        m_beg = ioff[m]; m_end = ioff[m + 1];
        a0 = mds[m]; n_m = mds[m + 1] - a0;
        L = s.ls_L[m];
        pl = item_plan(n_m, L);
        tabled = L <= CAND_CAP;
        if (tabled) {
          __syncwarp();
          const int e0 = geo.rowptr[m], e1 = geo.rowptr[m + 1];
          int cum = 0;
          for (int eb = e0; eb < e1; eb += 32) {
            const int e = eb + lane;
            int b0 = 0, n = 0;
            if (e < e1) { const int m2 = geo.col[e]; b0 = mds[m2]; n = mds[m2 + 1] - b0; }
            int inc = n;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
            const int off = cum + inc - n;
            for (int t = 0; t < n; ++t) cand[off + t] = b0 + t;        // a handful of MDs per connected module
            cum += __shfl_sync(0xffffffffu, inc, 31);
          }
          __syncwarp();
        }
      }
      const int row0 = (i - m_beg) * pl.rows_per_item;
      const int row1 = min(n_m, row0 + pl.rows_per_item);
      if (pl.S == 1) {
        const int W = pl.W, lw = lane & (W - 1), rs = lane / W;
        const bool vcol = lw < L;
        const int b = cand[min(lw, L - 1)];
        const Anchor B = load_anchor2(mpos, mcw, mmodt, b);
        const unsigned rowmask = (W == 32) ? 0xffffffffu : (((1u << W) - 1u) << (rs * W));
        for (int r0 = row0; r0 < row1; r0 += pl.R) {
          const int row = r0 + rs;
          const int a = a0 + min(row, n_m - 1);
          const Anchor A = load_anchor2(mpos, mcw, mmodt, a);
          float c = 0.f;
          const bool pass = vcol && row < row1 && ls_eval(A, B, c);
          const unsigned mask = __ballot_sync(0xffffffffu, pass);
          if (mask) {
            const unsigned rm = mask & rowmask;
            if (lw == 0 && row < row1 && rm) s.ls_start[a] = __popc(rm);
            if (pass) { LsRec rec; rec.a = a; rec.b = b; rec.rank = __popc(rm & lt); rec.c = c; stage[staged + __popc(mask & lt)] = rec; }
            staged += __popc(mask);
            __syncwarp();
            if (staged >= 32) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_LS, s.ls_rec, caps.max_ls, lane);
          }
        }
      } else {
        for (int row = row0; row < row1; ++row) {
          const int a = a0 + row;
          const Anchor A = load_anchor2(mpos, mcw, mmodt, a);
          int running = 0;
          for (int sw = 0; sw < pl.S; ++sw) {
            const int col = sw * 32 + lane;
            const int cc = min(col, L - 1);
            const int b = tabled ? cand[cc] : cand_walk(s, geo, m, cc);
            const Anchor B = load_anchor2(mpos, mcw, mmodt, b);
            float c = 0.f;
            const bool pass = col < L && ls_eval(A, B, c);
            const unsigned mask = __ballot_sync(0xffffffffu, pass);
            if (mask) {
              if (pass) { LsRec rec; rec.a = a; rec.b = b; rec.rank = running + __popc(mask & lt); rec.c = c; stage[staged + __popc(mask & lt)] = rec; }
              staged += __popc(mask);
              running += __popc(mask);
              __syncwarp();
              if (staged >= 32) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_LS, s.ls_rec, caps.max_ls, lane);
            }
          }
          if (lane == 0 && running) s.ls_start[a] = running;
        }
      }
    }
  }
  if (staged) flush_stage(stage, staged, s.cnt + LST_CNT_TMP_LS, s.ls_rec, caps.max_ls, lane);
}

__global__ void __launch_bounds__(256) k_ls_final(const Slot* __restrict__ slots, Caps caps) {
  const Slot& s = slots[blockIdx.y];
  const int n_rec = min(s.cnt[LST_CNT_TMP_LS], caps.max_ls);
  LST_FOR_ITEMS(i, n_rec) {
    const LsRec rec = s.ls_rec[i];
    const int pos = s.ls_start[rec.a] + rec.rank;
    if (pos < caps.max_ls) { s.ls_ab[pos] = make_int2(rec.a, rec.b); s.ls_c[pos] = rec.c; }
  }
}

}  // namespace lst
