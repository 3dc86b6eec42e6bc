// lst_pairs.cuh -- single-pass, order-preserving MD (a1) and LS (a2) kernels.
//
// Both stages test every cell of per-module rectangles (rows = inner objects of module m, columns = the
// module's candidate partners) and must emit the passing cells in the build order of SPEC.md 4.1-4.2
// (module, row, column).  The cells of all rectangles, in build order, form one flat index space (prefix scan
// of the per-module cell counts); one warp owns one *link* = a fixed-size range of that space:
//   1. prefilter:  all 32 lanes evaluate the cheap conservative form of the cuts (lst_math.cuh) on 32 cells;
//                  survivors (a few %) are appended, in order, to a per-warp queue in shared memory;
//   2. exact:      whenever the queue holds >= 32 cells a full warp evaluates the exact SPEC.md arithmetic
//                  on them; passing cells are appended, in order, to the warp's staging buffer;
//   3. place:      the link appends its objects (already in order) to an unordered per-slot record buffer and
//                  stores its count; a block scan over the link counts (k_scan) gives every link its base,
//                  and a per-link finalize warp copies the records to their final positions and writes the
//                  range tables (md_start / ls_start) of the rows the link owns.
// The output order depends only on the flat index, never on scheduling (bit-reproducible).  The staging
// buffer holds as many objects as a link has cells, so it cannot overflow.
// Capacity overflow: the record buffer (same capacity as the stage) may then have dropped records of early
// links, so the CHAIN instantiation re-runs the stage: links are handed out by an atomic ticket, each obtains
// the count of all earlier links by decoupled look-back and writes its first objects in place (a link only
// waits for links that are already running: no deadlock).  It returns at once unless the overflow bit is set
// (in-place waiting behind slow links makes it ~4x slower than the record path, measured r01).
#pragma once
#include "lst_kernels.cuh"

namespace lst {

constexpr int PAIR_WARPS = 4;        // warps per block
constexpr int Q_CAP = 64;            // survivor queue per warp (drained at >= 32)
constexpr int MD_WIN = 32;           // modules of a link cached in shared memory (one per lane)

__device__ __forceinline__ unsigned lanemask_lt() { unsigned m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

// ---- decoupled look-back over 64-bit status words: flag (2 bits) | run epoch (30 bits) | value (32 bits).
// A word counts only if its epoch is the current run's (k_hist, the first kernel of a run, increments the slot's
// device-side run counter), so the status arrays never need clearing and the launch sequence has no per-run
// arguments (it can be replayed as a CUDA graph).
constexpr unsigned long long CH_AGG = 1ull << 62, CH_INC = 2ull << 62, CH_VAL = 0xFFFFFFFFull;
__device__ __forceinline__ unsigned chain_flag(unsigned long long w, unsigned epoch) {
  return (((unsigned)(w >> 32)) & 0x3FFFFFFFu) == epoch ? (unsigned)(w >> 62) : 0u;
}
__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// exclusive prefix of `count` over links [0, link); called by all 32 lanes, publishes the inclusive prefix
__device__ __forceinline__ int chain_exclusive(unsigned long long* st, int link, int count, int lane, unsigned epoch) {
  const unsigned long long ep = (unsigned long long)epoch << 32;
  if (link == 0) {
    if (lane == 0) st_status(st, CH_INC | ep | (unsigned long long)(unsigned)count);
    return 0;
  }
  if (lane == 0) st_status(st + link, CH_AGG | ep | (unsigned long long)(unsigned)count);
  int excl = 0;
  int idx = link - 1 - lane;
  while (true) {
    unsigned long long w;
    unsigned fl;
    do {
      w = (idx >= 0) ? ld_status(st + idx) : (CH_INC | ep);
      fl = chain_flag(w, epoch);
    } while (__any_sync(0xffffffffu, fl == 0u));
    const unsigned inc = __ballot_sync(0xffffffffu, fl == 2u);
    const int first = inc ? (__ffs(inc) - 1) : 31;     // nearest predecessor that holds an inclusive prefix
    int v = (lane <= first) ? (int)(w & CH_VAL) : 0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    excl += v;
    if (inc) break;
    idx -= 32;
  }
  if (lane == 0) st_status(st + link, CH_INC | ep | (unsigned long long)(unsigned)(excl + count));
  return excl;
}

__device__ __forceinline__ int warp_ticket(int* counter, int lane) {
  int t = 0;
  if (lane == 0) t = atomicAdd(counter, 1);
  return __shfl_sync(0xffffffffu, t, 0);
}


// first index i in [0, n] with off[i] > x (off non-decreasing); n + 1 if none
__device__ __forceinline__ int upper_bound_g(const int* __restrict__ off, int n, int x) {
  int lo = 0, hi = n + 1;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (off[mid] > x) hi = mid; else lo = mid + 1;
  }
  return lo;
}
// largest m in [mS, mE] with off[m] <= f (exists by construction); among equal offsets the last one, i.e. the
// module that really owns cell f
__device__ __forceinline__ int owner_module(const int* __restrict__ off, int mS, int mE, int f) {
  int lo = mS, hi = mE;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (off[mid] <= f) lo = mid; else hi = mid - 1;
  }
  return lo;
}
__device__ __forceinline__ int lower_bound_s(const int* a, int n, int x) {   // first i with a[i] >= x
  int lo = 0, hi = n;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] < x) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ void divmod_small(int v, int d, int& q, int& r) {   // 0 <= v < 2^22, d > 0
  q = (int)(((float)v + 0.5f) * rcp_fast((float)d));
  r = v - q * d;
  if (r < 0) { --q; r += d; } else if (r >= d) { ++q; r -= d; }
}

// ------------------------------------------------------------------------------------------------
// a1: cells = (lower hit i, upper hit j) of module m, flat index md_pair_off[m] + i*n_up + j
// ------------------------------------------------------------------------------------------------
struct MdWarp {   // per-warp shared memory
  int w_off[MD_WIN + 1], w_lb[MD_WIN], w_ub[MD_WIN], w_nup[MD_WIN], w_mt[MD_WIN];   // the link's first modules
  int q_lo[Q_CAP], q_up[Q_CAP], q_mt[Q_CAP], q_f[Q_CAP];
  int p_lo[MD_LP], p_up[MD_LP], p_mt[MD_LP], p_f[MD_LP];
  float p_c[MD_LP], p_w[MD_LP];
};

// exact evaluation of `n` (<= 32) queued cells; appends the passing ones in order; returns the new count
__device__ __forceinline__ int md_drain(const Slot& s, MdWarp& W, int n, int pn, int lane, unsigned lt) {
  bool pass = false;
  int p_lo = 0, p_up = 0, mtm = 0, f = 0;
  float c = 0.f, w = 0.f;
  if (lane < n) {
    p_lo = W.q_lo[lane]; p_up = W.q_up[lane]; mtm = W.q_mt[lane]; f = W.q_f[lane];
    const float4 h1 = s.hit[p_lo], h2 = s.hit[p_up];
    pass = md_eval(h1.x, h1.y, h1.z, h1.w, h2.x, h2.y, h2.z, h2.w, mtm & 3, c, w);
  }
  const unsigned mask = __ballot_sync(0xffffffffu, pass);
  if (pass) {
    const int i = pn + __popc(mask & lt);
    W.p_lo[i] = p_lo; W.p_up[i] = p_up; W.p_mt[i] = mtm; W.p_f[i] = f; W.p_c[i] = c; W.p_w[i] = w;
  }
  return pn + __popc(mask);
}

template <bool CHAIN>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_md_links(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  __shared__ MdWarp Wall[PAIR_WARPS];
  const Slot& s = slots[blockIdx.y];
  const unsigned epoch = *s.epoch_dev;
  if (CHAIN && !(s.cnt[CNT_STATUS] & LST_ST_OVF_MD)) return;
  const int lane = threadIdx.x & 31;
  MdWarp& W = Wall[threadIdx.x >> 5];
  const unsigned lt = lanemask_lt();
  const int M = geo.n_modules;
  const int* __restrict__ off = s.md_pair_off;
  const int* __restrict__ ss = s.sensor_start;
  const float4* __restrict__ hit = s.hit;
  const int total_cells = min(off[M], MAX_CELLS);       // beyond: flagged by the scan that made `off`
  const int n_links = total_cells / MD_LP + 1;
  const int cap = caps.max_md;
  int link;
  while (true) {      // links are handed out dynamically: their cost varies with the number of modules they span
    link = warp_ticket(s.cnt + (CHAIN ? LST_CNT_TICKET_MD : LST_CNT_DYN_MD), lane);
    if (link >= n_links) break;
    const int lo = link * MD_LP, hi = min(total_cells, lo + MD_LP);
    int qn = 0, pn = 0;
    if (lo < hi) {
      // cache the first MD_WIN modules of the link (normally all of them)
      const int mS = s.md_link_mod[link];
      __syncwarp();
      {
        const int m = mS + lane;
        int o = 0x7fffffff, lb = 0, ub = 0, ue = 0, mt = 0;
        if (m < M) { o = off[m]; lb = ss[2 * m]; ub = ss[2 * m + 1]; ue = ss[2 * m + 2]; mt = geo.modt[m]; }
        W.w_off[lane] = o; W.w_lb[lane] = lb; W.w_ub[lane] = ub; W.w_nup[lane] = ue - ub; W.w_mt[lane] = (m << 2) | mt;
        if (lane == 0) W.w_off[MD_WIN] = (mS + MD_WIN <= M) ? off[mS + MD_WIN] : 0x7fffffff;
      }
      __syncwarp();
      const int win_end = W.w_off[MD_WIN];
      for (int f0 = lo; f0 < hi; f0 += 32) {
        const int f = f0 + lane;
        bool pre = false;
        int p_lo = 0, p_up = 0, mtm = 0;
        if (f < hi) {
          int loc, lb, ub, nup;
          if (f < win_end) {
            int k = 0;
#pragma unroll
            for (int step = MD_WIN / 2; step > 0; step >>= 1)
              if (W.w_off[k + step] <= f) k += step;
            loc = f - W.w_off[k]; lb = W.w_lb[k]; ub = W.w_ub[k]; nup = W.w_nup[k]; mtm = W.w_mt[k];
          } else {     // sparse region: the link spans more than MD_WIN modules
            const int m = owner_module(off, mS + MD_WIN, M - 1, f);
            loc = f - off[m]; lb = ss[2 * m]; ub = ss[2 * m + 1]; nup = ss[2 * m + 2] - ub; mtm = (m << 2) | geo.modt[m];
          }
          int i, j;
          divmod_small(loc, nup, i, j);
          p_lo = lb + i; p_up = ub + j;
          const float4 h1 = __ldg(hit + p_lo), h2 = __ldg(hit + p_up);
          pre = md_prefilter(h1.x, h1.y, h1.z, h1.w, h2.x, h2.y, h2.z, h2.w, mtm & 3);
        }
        const unsigned mask = __ballot_sync(0xffffffffu, pre);
        if (mask) {
          if (pre) { const int i = qn + __popc(mask & lt); W.q_lo[i] = p_lo; W.q_up[i] = p_up; W.q_mt[i] = mtm; W.q_f[i] = f - lo; }
          qn += __popc(mask);
          __syncwarp();
          if (qn >= 32) {
            pn = md_drain(s, W, 32, pn, lane, lt);
            __syncwarp();
            const int rest = qn - 32;
            int a = 0, b = 0, c = 0, d = 0;
            if (lane < rest) { a = W.q_lo[32 + lane]; b = W.q_up[32 + lane]; c = W.q_mt[32 + lane]; d = W.q_f[32 + lane]; }
            __syncwarp();
            if (lane < rest) { W.q_lo[lane] = a; W.q_up[lane] = b; W.q_mt[lane] = c; W.q_f[lane] = d; }
            qn = rest;
            __syncwarp();
          }
        }
      }
      if (qn) pn = md_drain(s, W, qn, pn, lane, lt);
      __syncwarp();
    }
    if (!CHAIN) {      // append the link's MDs to the record buffer, remember where and how many
      int soff = 0;
      if (lane == 0) { soff = pn ? atomicAdd(s.cnt + LST_CNT_FILL_MD, pn) : 0; s.md_link_cnt[link] = pn; s.md_link_soff[link] = soff; }
      soff = __shfl_sync(0xffffffffu, soff, 0);
      for (int i = lane; i < pn; i += 32)
        if (soff + i < cap) {
          MdRec r; r.p_lo = W.p_lo[i]; r.p_up = W.p_up[i]; r.mtm = W.p_mt[i]; r.f = W.p_f[i]; r.c = W.p_c[i]; r.w = W.p_w[i]; r.link = link; r.pad = 0;
          s.md_rec[soff + i] = r;
        }
      __syncwarp();
      continue;
    }
    // CHAIN (overflow re-run): base by look-back, objects and range table written in place
    const int base = chain_exclusive(s.chain_md, link, pn, lane, epoch);
    for (int i = lane; i < pn; i += 32) {
      const int pos = base + i;
      if (pos < cap) {
        const int p_lo = W.p_lo[i], p_up = W.p_up[i];
        s.md_hits[pos] = make_int2(s.hit_orig[p_lo], s.hit_orig[p_up]);
        s.md_modt[pos] = W.p_mt[i];
        s.md_pos[pos] = hit[p_lo];              // (x, y, z, r1)
        s.md_cw[pos] = make_float2(W.p_c[i], W.p_w[i]);
        s.md_aux[pos] = make_float4(W.p_c[i], W.p_w[i], md_relf(W.p_mt[i] & 3), 0.f);
      }
    }
    int sr = 0;
    if (lane < 2) sr = upper_bound_g(off, M, lane == 0 ? lo - 1 : lo + MD_LP - 1);
    const int mOwn0 = __shfl_sync(0xffffffffu, sr, 0), mOwn1 = min(M, __shfl_sync(0xffffffffu, sr, 1));
    for (int m = mOwn0 + lane; m < mOwn1; m += 32) s.md_start[m] = min(base + lower_bound_s(W.p_f, pn, off[m] - lo), cap);
    if (link == n_links - 1 && lane == 0) {
      const int total = base + pn;
      s.md_start[M] = min(total, cap);
      s.cnt[LST_CNT_MD] = min(total, cap);
      s.cnt[LST_CNT_RAW_MD] = total;
    }
    __syncwarp();
  }
}

// a1 finalize (md_link_cnt holds the exclusive scan of the link counts by now): one thread per record copies it
// to base[link] + its index inside the link; one thread per module writes md_start[m] = number of MDs before the
// module's first cell
__global__ void __launch_bounds__(256) k_md_final(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  const Slot& s = slots[blockIdx.y];
  if (s.cnt[CNT_STATUS] & LST_ST_OVF_MD) return;       // the CHAIN pass rewrites the stage
  const int M = geo.n_modules;
  const int* __restrict__ off = s.md_pair_off;
  const int* __restrict__ base = s.md_link_cnt;
  const int* __restrict__ soff = s.md_link_soff;
  const int n_rec = min(s.cnt[LST_CNT_FILL_MD], caps.max_md);
  LST_FOR_ITEMS(j, n_rec) {
    const MdRec r = s.md_rec[j];
    const int pos = base[r.link] + (j - soff[r.link]);
    s.md_hits[pos] = make_int2(s.hit_orig[r.p_lo], s.hit_orig[r.p_up]);
    s.md_modt[pos] = r.mtm;
    s.md_pos[pos] = s.hit[r.p_lo];
    s.md_cw[pos] = make_float2(r.c, r.w);
    s.md_aux[pos] = make_float4(r.c, r.w, md_relf(r.mtm & 3), 0.f);     // (c, w, f, -): one load for the LS prefilter
  }
  const int total_cells = min(off[M], MAX_CELLS);
  LST_FOR_ITEMS(m, M + 1) {
    const int x = min(off[m], total_cells);
    const int link = x / MD_LP, rel = x - link * MD_LP;
    const int b = base[link], pn = base[link + 1] - b;
    const MdRec* __restrict__ rec = s.md_rec + soff[link];
    int l = 0, h = pn;
    while (l < h) { const int mid = (l + h) >> 1; if (rec[mid].f < rel) l = mid + 1; else h = mid; }
    s.md_start[m] = b + l;
  }
}

// ------------------------------------------------------------------------------------------------
// a2: cells = (MD a of module m, candidate column) with flat index ls_off[m] + row*L[m] + col; the columns of m
// are the MDs of its CSR-connected modules in ascending MD index (L[m] of them, listed in ls_cand)
// ------------------------------------------------------------------------------------------------
// plan, three small launches: (1) candidate count L[m] and cell count n_m * L[m] per module; (2) one block per
// event: exclusive scans of the cell counts and of the candidate-table offsets, link -> module table; (3) the
// candidate table itself
__global__ void __launch_bounds__(256) k_ls_plan1(const Slot* __restrict__ slots, Geo geo) {
  const Slot& s = slots[blockIdx.y];
  const int* __restrict__ mds = s.md_start;
  LST_FOR_ITEMS(m, geo.n_modules) {
    const int n_m = mds[m + 1] - mds[m];
    int L = 0;
    if (n_m > 0) {
      const int e1 = geo.rowptr[m + 1];
      for (int e = geo.rowptr[m]; e < e1; ++e) { const int m2 = geo.col[e]; L += mds[m2 + 1] - mds[m2]; }
    }
    long long cells = (long long)n_m * L;
    if (cells > MAX_CELLS) {      // beyond any event the capacities admit: drop the module's cells, flag the stage
      cells = 0; L = 0;
      atomicOr(reinterpret_cast<unsigned*>(s.cnt + CNT_STATUS), LST_ST_OVF_LS);
    }
    s.ls_L[m] = L;
    s.ls_off[m] = (int)cells;
    s.ls_coff[m] = L;
  }
}
__global__ void __launch_bounds__(SCAN_THREADS) k_ls_plan2(const Slot* __restrict__ slots, Geo geo) {
  __shared__ int sm[34];
  const Slot& s = slots[blockIdx.y];
  const int M = geo.n_modules;
  const int total = block_scan_inplace(s.ls_off, M, 0x7fffffff, sm);
  __syncthreads();
  block_scan_inplace(s.ls_coff, M, 0x7fffffff, sm);
  __syncthreads();
  if (threadIdx.x == 0 && total > MAX_CELLS) atomicOr(reinterpret_cast<unsigned*>(s.cnt + CNT_STATUS), LST_ST_OVF_LS);
  link_owner_table(s.ls_off, M, LS_LP, s.ls_link_mod);
}
__global__ void __launch_bounds__(256) k_ls_plan3(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  const Slot& s = slots[blockIdx.y];
  const int* __restrict__ mds = s.md_start;
  const int cand_cap = CAND_PER_MD * caps.max_md;
  const int lane = threadIdx.x & 31;
  // one warp per module: the lanes take the CSR entries, a warp scan places each entry's MD range
  for (int m = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; m < geo.n_modules; m += (gridDim.x * blockDim.x) >> 5) {
    const int L = s.ls_L[m];
    int o = s.ls_coff[m];
    if (L == 0 || o + L > cand_cap) continue;        // modules beyond the table walk the CSR row instead
    const int e0 = geo.rowptr[m], e1 = geo.rowptr[m + 1];
    for (int eb = e0; eb < e1; eb += 32) {
      const int e = eb + lane;
      int b0 = 0, n = 0;
      if (e < e1) { const int m2 = geo.col[e]; b0 = mds[m2]; n = mds[m2 + 1] - b0; }
      int inc = n;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
      const int w = o + inc - n;
      for (int t = 0; t < n; ++t) s.ls_cand[w + t] = b0 + t;
      o += __shfl_sync(0xffffffffu, inc, 31);
    }
  }
}

struct LsWarp {
  int w_off[MD_WIN + 1], w_a0[MD_WIN], w_L[MD_WIN], w_co[MD_WIN];      // the link's next modules
  int q_a[Q_CAP], q_b[Q_CAP], q_f[Q_CAP];
  int p_a[LS_LP], p_b[LS_LP], p_f[LS_LP];
  float p_c[LS_LP];
};

__device__ __forceinline__ Anchor load_anchor(const Slot& s, int i) {
  const float4 p = s.md_pos[i];
  const float2 q = s.md_cw[i];
  Anchor a; a.x = p.x; a.y = p.y; a.z = p.z; a.r = p.w; a.c = q.x; a.w = q.y; a.mt = s.md_modt[i] & 3;
  return a;
}

// column -> MD index by walking the CSR row (only for modules beyond the candidate table)
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

__device__ __forceinline__ int ls_drain(const Slot& s, LsWarp& W, int n, int pn, int lane, unsigned lt) {
  bool pass = false;
  int a = 0, b = 0, f = 0;
  float c = 0.f;
  if (lane < n) {
    a = W.q_a[lane]; b = W.q_b[lane]; f = W.q_f[lane];
    const Anchor A = load_anchor(s, a), B = load_anchor(s, b);
    pass = ls_eval(A, B, c);
  }
  const unsigned mask = __ballot_sync(0xffffffffu, pass);
  if (pass) {
    const int i = pn + __popc(mask & lt);
    W.p_a[i] = a; W.p_b[i] = b; W.p_f[i] = f; W.p_c[i] = c;
  }
  return pn + __popc(mask);
}

// append the survivors of one sweep to the queue (in lane order); a full warp of queued cells is evaluated at once
__device__ __forceinline__ void ls_push(const Slot& s, LsWarp& W, bool pre, int a, int b, int f, int& qn, int& pn, int lane, unsigned lt) {
  const unsigned mask = __ballot_sync(0xffffffffu, pre);
  if (!mask) return;
  if (pre) { const int i = qn + __popc(mask & lt); W.q_a[i] = a; W.q_b[i] = b; W.q_f[i] = f; }
  qn += __popc(mask);
  __syncwarp();
  if (qn >= 32) {
    pn = ls_drain(s, W, 32, pn, lane, lt);
    __syncwarp();
    const int rest = qn - 32;
    int x = 0, y = 0, z = 0;
    if (lane < rest) { x = W.q_a[32 + lane]; y = W.q_b[32 + lane]; z = W.q_f[32 + lane]; }
    __syncwarp();
    if (lane < rest) { W.q_a[lane] = x; W.q_b[lane] = y; W.q_f[lane] = z; }
    qn = rest;
    __syncwarp();
  }
}

// first MD index whose row starts at a flat position >= x (rows are in MD order, positions non-decreasing)
__device__ __forceinline__ int first_row_at(const Slot& s, const int* __restrict__ off, int M, int x) {
  const int* __restrict__ mds = s.md_start;
  if (x > off[M]) return mds[M];
  const int mB = (x <= 0) ? 0 : upper_bound_g(off, M, x - 1);     // first module with off[m] >= x (<= M)
  if (mB > 0) {
    const int mP = mB - 1, L = s.ls_L[mP];                        // off[mP] < x: its later rows may still start >= x
    if (L > 0) {
      const int n_m = mds[mP + 1] - mds[mP];
      const int r0 = (x - off[mP] + L - 1) / L;
      if (r0 < n_m) return mds[mP] + r0;
    }
  }
  return mds[mB];
}

template <bool CHAIN>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_ls_links(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  __shared__ LsWarp Wall[PAIR_WARPS];
  const Slot& s = slots[blockIdx.y];
  const unsigned epoch = *s.epoch_dev;
  if (CHAIN && !(s.cnt[CNT_STATUS] & LST_ST_OVF_LS)) return;
  const int lane = threadIdx.x & 31;
  LsWarp& W = Wall[threadIdx.x >> 5];
  const unsigned lt = lanemask_lt();
  const int M = geo.n_modules;
  const int* __restrict__ off = s.ls_off;
  const int* __restrict__ mds = s.md_start;
  const int* __restrict__ cand = s.ls_cand;
  const float4* __restrict__ mpos = s.md_pos;
  const float4* __restrict__ maux = s.md_aux;
  const int total_cells = min(off[M], MAX_CELLS);
  const int n_links = total_cells / LS_LP + 1;
  const int cap = caps.max_ls, cand_cap = CAND_PER_MD * caps.max_md;
  int link;
  while (true) {
    link = warp_ticket(s.cnt + (CHAIN ? LST_CNT_TICKET_LS : LST_CNT_DYN_LS), lane);
    if (link >= n_links) break;
    const int lo = link * LS_LP, hi = min(total_cells, lo + LS_LP);
    int qn = 0, pn = 0;
    if (lo < hi) {
      int mW = s.ls_link_mod[link];      // module that owns the next unprocessed cell
      int fc = lo;                       // next unprocessed cell
      while (fc < hi) {
        // cache the next MD_WIN modules (offsets, first MD, candidate count, candidate-table offset)
        __syncwarp();
        {
          const int m = mW + lane;
          int o = 0x7fffffff, a0 = 0, L = 1, co = 0;
          if (m < M) { o = off[m]; a0 = mds[m]; L = s.ls_L[m]; co = s.ls_coff[m]; }
          W.w_off[lane] = o; W.w_a0[lane] = a0; W.w_L[lane] = L; W.w_co[lane] = co;
          if (lane == 0) W.w_off[MD_WIN] = (mW + MD_WIN <= M) ? off[mW + MD_WIN] : 0x7fffffff;
        }
        __syncwarp();
        const int end = min(hi, W.w_off[MD_WIN]);
        if (W.w_off[1] >= hi) {
          // dense: the rest of the link lies in one module -- (row, col) advance incrementally
          const int om = W.w_off[0], a0 = W.w_a0[0], L = W.w_L[0], co = W.w_co[0];
          const bool tabled = co + L <= cand_cap;
          const int c0 = fc - om, c1 = hi - om;
          int row, col, q32, r32;                       // the lane's cell (row, col); 32 cells further = (+q32, +r32)
          divmod_small(c0 + lane, L, row, col);
          divmod_small(32, L, q32, r32);
          for (int cb = c0; cb < c1; cb += 32) {
            const int cell = cb + lane;
            bool pre = false;
            int a = 0, b = 0;
            if (cell < c1) {
              a = a0 + row;
              b = tabled ? __ldg(cand + co + col) : cand_walk(s, geo, mW, col);
              pre = ls_prefilter(__ldg(mpos + a), __ldg(maux + a), __ldg(mpos + b), __ldg(maux + b));
            }
            row += q32; col += r32;
            if (col >= L) { col -= L; ++row; }
            ls_push(s, W, pre, a, b, om + cell - lo, qn, pn, lane, lt);
          }
          fc = hi;
        } else {
          // several modules: every lane finds the module of its cell in the cached window
          for (int f0 = fc; f0 < end; f0 += 32) {
            const int f = f0 + lane;
            bool pre = false;
            int a = 0, b = 0;
            if (f < end) {
              int k = 0;
#pragma unroll
              for (int step = MD_WIN / 2; step > 0; step >>= 1)
                if (W.w_off[k + step] <= f) k += step;
              const int L = W.w_L[k], co = W.w_co[k];
              int row, col;
              divmod_small(f - W.w_off[k], L, row, col);
              a = W.w_a0[k] + row;
              b = (co + L <= cand_cap) ? __ldg(cand + co + col) : cand_walk(s, geo, mW + k, col);
              pre = ls_prefilter(__ldg(mpos + a), __ldg(maux + a), __ldg(mpos + b), __ldg(maux + b));
            }
            ls_push(s, W, pre, a, b, f - lo, qn, pn, lane, lt);
          }
          fc = end;
          mW += MD_WIN;          // off[mW + MD_WIN] <= fc: the owner of cell fc is at or after it
        }
      }
      if (qn) pn = ls_drain(s, W, qn, pn, lane, lt);
      __syncwarp();
    }
    if (!CHAIN) {
      int soff = 0;
      if (lane == 0) { soff = pn ? atomicAdd(s.cnt + LST_CNT_FILL_LS, pn) : 0; s.ls_link_cnt[link] = pn; s.ls_link_soff[link] = soff; }
      soff = __shfl_sync(0xffffffffu, soff, 0);
      for (int i = lane; i < pn; i += 32)
        if (soff + i < cap) { LsRec r; r.a = W.p_a[i]; r.b = W.p_b[i]; r.lf = (link << LS_LP_BITS) | W.p_f[i]; r.c = W.p_c[i]; s.ls_rec[soff + i] = r; }
      __syncwarp();
      continue;
    }
    const int base = chain_exclusive(s.chain_ls, link, pn, lane, epoch);
    for (int i = lane; i < pn; i += 32)
      if (base + i < cap) { s.ls_ab[base + i] = make_int2(W.p_a[i], W.p_b[i]); s.ls_c[base + i] = W.p_c[i]; }
    // LSs whose inner MD is a = [ls_start[a], ls_start[a+1]): the link owns the rows that start in its range
    int sr = 0;
    if (lane < 2) sr = first_row_at(s, off, M, lane == 0 ? lo : lo + LS_LP);
    const int aLo = __shfl_sync(0xffffffffu, sr, 0), aHi = __shfl_sync(0xffffffffu, sr, 1);
    for (int a = aLo + lane; a < aHi; a += 32) {
      const int m = s.md_modt[a] >> 2;
      const int rel = off[m] + (a - mds[m]) * s.ls_L[m] - lo;
      s.ls_start[a] = min(base + lower_bound_s(W.p_f, pn, rel), cap);
    }
    if (link == n_links - 1 && lane == 0) {
      const int total = base + pn;
      s.ls_start[mds[M]] = min(total, cap);
      s.cnt[LST_CNT_LS] = min(total, cap);
      s.cnt[LST_CNT_RAW_LS] = total;
    }
    __syncwarp();
  }
}

// a2 finalize: one thread per record; one thread per MD row for ls_start
__global__ void __launch_bounds__(256) k_ls_final(const Slot* __restrict__ slots, Geo geo, Caps caps) {
  const Slot& s = slots[blockIdx.y];
  if (s.cnt[CNT_STATUS] & LST_ST_OVF_LS) return;
  const int M = geo.n_modules;
  const int* __restrict__ off = s.ls_off;
  const int* __restrict__ mds = s.md_start;
  const int* __restrict__ base = s.ls_link_cnt;
  const int* __restrict__ soff = s.ls_link_soff;
  const int n_rec = min(s.cnt[LST_CNT_FILL_LS], caps.max_ls);
  LST_FOR_ITEMS(j, n_rec) {
    const LsRec r = s.ls_rec[j];
    const int link = r.lf >> LS_LP_BITS;
    const int pos = base[link] + (j - soff[link]);
    s.ls_ab[pos] = make_int2(r.a, r.b);
    s.ls_c[pos] = r.c;
  }
  const int total_cells = min(off[M], MAX_CELLS);
  const int n_md = mds[M];
  LST_FOR_ITEMS(a, n_md + 1) {
    int x = total_cells;
    if (a < n_md) { const int m = s.md_modt[a] >> 2; x = min(off[m] + (a - mds[m]) * s.ls_L[m], total_cells); }
    const int link = x >> LS_LP_BITS, rel = x - (link << LS_LP_BITS);
    const int b = base[link], pn = base[link + 1] - b;
    const LsRec* __restrict__ rec = s.ls_rec + soff[link];
    int l = 0, h = pn;
    while (l < h) { const int mid = (l + h) >> 1; if ((rec[mid].lf & (LS_LP - 1)) < rel) l = mid + 1; else h = mid; }
    s.ls_start[a] = b + l;
  }
}

}  // namespace lst
