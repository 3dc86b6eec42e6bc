// lst_tuples.cuh -- a3 (triplets) and a4 (quintuplet candidates), single pass, build order preserved.
//
// One thread owns one inner object (first LS / inner T3) and loops over its few partners (about one on average).
// A block takes a tile of TUPLE_TPB consecutive rows by atomic ticket, evaluates them once (up to TUPLE_STASH
// passing partners per row stay in registers), scans the row counts, obtains the number of objects of all earlier
// tiles by decoupled look-back (lst_pairs.cuh) and writes its objects at their final positions.  Tiles are uniform
// (unlike the a1/a2 links), so nobody waits long; tickets make a tile wait only for tiles that already run.
// Capacity overflow: positions >= cap are not written, the last tile records the unclamped total and the flag.
#pragma once
#include "lst_pairs.cuh"

namespace lst {

constexpr int TUPLE_TPB = 128, TUPLE_STASH = 3;

// block-wide exclusive scan of one int per thread (TUPLE_TPB threads); returns the exclusive prefix, total in `total`
__device__ __forceinline__ int block_excl(int v, int* sm /*[TUPLE_TPB/32 + 1]*/, int& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
  if (lane == 31) sm[wid] = inc;
  __syncthreads();
  int wbase = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < TUPLE_TPB / 32; ++w) { const int c = sm[w]; if (w < wid) wbase += c; tot += c; }
  total = tot;
  __syncthreads();
  return wbase + inc - v;
}

// a3 (SPEC.md 4.3): rows = LS l0 = (a,b); partners = LSs whose inner MD is b
__global__ void __launch_bounds__(TUPLE_TPB) k_t3_one(const Slot* __restrict__ slots, Caps caps) {
  pdl_begin();
  __shared__ int sm[TUPLE_TPB / 32 + 1];
  __shared__ int s_tile, s_base;
  const Slot& s = slots[blockIdx.y];
  const unsigned epoch = *s.epoch_dev;
  const int n = s.cnt[LST_CNT_LS];
  const int n_tiles = (n + TUPLE_TPB - 1) / TUPLE_TPB + (n == 0);
  const int cap = caps.max_t3;
  while (true) {
    if (threadIdx.x == 0) s_tile = atomicAdd(s.cnt + LST_CNT_DYN_T3, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int l0 = tile * TUPLE_TPB + threadIdx.x;
    int np = 0;
    int st_j[TUPLE_STASH], st_c[TUPLE_STASH];
    float st_k[TUPLE_STASH];
    int2 ab = make_int2(0, 0);
    int j0 = 0, j1 = 0;
    Pt A{}, B{};
    float c0 = 0.f;
    if (l0 < n) {
      ab = s.ls_ab[l0];
      j0 = s.ls_start[ab.y]; j1 = s.ls_start[ab.y + 1];
      if (j0 < j1) {
        A = make_pt(s.md_pos[ab.x], s.md_modt[ab.x] & 3);
        B = make_pt(s.md_pos[ab.y], s.md_modt[ab.y] & 3);
        c0 = s.ls_c[l0];
        // partners one and two steps ahead are in flight while the current one is evaluated (index, then its MD)
        int cn = s.ls_ab[j0].y, cnn = (j0 + 1 < j1) ? s.ls_ab[j0 + 1].y : 0;
        float4 pn = s.md_pos[cn];
        int mn = s.md_modt[cn];
        float ln = s.ls_c[j0];
        for (int j = j0; j < j1; ++j) {
          const int cidx = cn;
          const Pt C = make_pt(pn, mn & 3);
          const float lcj = ln;
          if (j + 1 < j1) {
            cn = cnn; pn = s.md_pos[cn]; mn = s.md_modt[cn]; ln = s.ls_c[j + 1];
            if (j + 2 < j1) cnn = s.ls_ab[j + 2].y;
          }
          float k;
          if (!triplet_eval(A, B, C, k)) continue;
          if (!(fabsf(fs(c0, k)) <= LST_C_TOL3)) continue;                                  // T3
          if (!(fabsf(fs(lcj, k)) <= LST_C_TOL3)) continue;
#pragma unroll
          for (int q = 0; q < TUPLE_STASH; ++q)
            if (np == q) { st_j[q] = j; st_c[q] = cidx; st_k[q] = k; }
          ++np;
        }
      }
    }
    int block_total;
    const int excl = block_excl(np, sm, block_total);
    if (threadIdx.x < 32) {
      const int b = chain_exclusive(s.chain_t3, tile, block_total, threadIdx.x, epoch);
      if (threadIdx.x == 0) s_base = b;
    }
    __syncthreads();
    const int base = s_base;
    if (l0 < n) {
      int pos = base + excl;
      s.t3_off[l0] = min(pos, cap);
      if (np <= TUPLE_STASH) {
#pragma unroll
        for (int q = 0; q < TUPLE_STASH; ++q)
          if (q < np && pos + q < cap) { s.t3_abc[pos + q] = make_int4(ab.x, ab.y, st_c[q], l0); s.t3_l1[pos + q] = st_j[q]; s.t3_k[pos + q] = st_k[q]; }
      } else {            // more partners than the stash holds: evaluate the row again
        for (int j = j0; j < j1; ++j) {
          const int cidx = s.ls_ab[j].y;
          const Pt C = make_pt(s.md_pos[cidx], s.md_modt[cidx] & 3);
          float k;
          if (!triplet_eval(A, B, C, k)) continue;
          if (!(fabsf(fs(c0, k)) <= LST_C_TOL3)) continue;
          if (!(fabsf(fs(s.ls_c[j], k)) <= LST_C_TOL3)) continue;
          if (pos < cap) { s.t3_abc[pos] = make_int4(ab.x, ab.y, cidx, l0); s.t3_l1[pos] = j; s.t3_k[pos] = k; }
          ++pos;
        }
      }
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
      const int total = base + block_total;
      s.t3_off[n] = min(total, cap);
      s.cnt[LST_CNT_T3] = min(total, cap);
      s.cnt[LST_CNT_RAW_T3] = total;
      if (total > cap) atomicOr(reinterpret_cast<unsigned*>(s.cnt + CNT_STATUS), LST_ST_OVF_T3);
    }
    __syncthreads();
  }
}

// a4 (SPEC.md 4.4): rows = T3 u = (a,b,c); partners = T3s whose inner MD is c; the bridge (b,c,d) must pass
__global__ void __launch_bounds__(TUPLE_TPB) k_t5_one(const Slot* __restrict__ slots, Caps caps) {
  pdl_begin();
  __shared__ int sm[TUPLE_TPB / 32 + 1];
  __shared__ int s_tile, s_base;
  const Slot& s = slots[blockIdx.y];
  const unsigned epoch = *s.epoch_dev;
  const int n = s.cnt[LST_CNT_T3];
  const int n_tiles = (n + TUPLE_TPB - 1) / TUPLE_TPB + (n == 0);
  const int cap = caps.max_t5c;
  // T3s whose inner MD is a = [t3_start[a], t3_start[a+1]) with t3_start[a] = t3_off[ls_start[a]]: the table is an output
  // (lst_get); this kernel itself goes through t3_off / ls_start so that it need not wait for it
  while (true) {
    if (threadIdx.x == 0) s_tile = atomicAdd(s.cnt + LST_CNT_DYN_T5, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int u = tile * TUPLE_TPB + threadIdx.x;
    int np = 0;
    int st_v[TUPLE_STASH];
    float st_k[TUPLE_STASH];
    int4 abc = make_int4(0, 0, 0, 0);
    int v0 = 0, v1 = 0;
    Pt B{}, C{};
    if (u < n) {
      abc = s.t3_abc[u];
      v0 = s.t3_off[s.ls_start[abc.z]]; v1 = s.t3_off[s.ls_start[abc.z + 1]];
      if (v0 < v1) {
        B = make_pt(s.md_pos[abc.y], s.md_modt[abc.y] & 3);
        C = make_pt(s.md_pos[abc.z], s.md_modt[abc.z] & 3);
        int dn = s.t3_abc[v0].y, dnn = (v0 + 1 < v1) ? s.t3_abc[v0 + 1].y : 0;           // partners ahead in flight, as in a3
        float4 pn = s.md_pos[dn];
        int mn = s.md_modt[dn];
        for (int v = v0; v < v1; ++v) {
          const Pt D = make_pt(pn, mn & 3);
          if (v + 1 < v1) {
            dn = dnn; pn = s.md_pos[dn]; mn = s.md_modt[dn];
            if (v + 2 < v1) dnn = s.t3_abc[v + 2].y;
          }
          float kbr;
          if (!triplet_eval(B, C, D, kbr)) continue;                                        // Q1, Q2
#pragma unroll
          for (int q = 0; q < TUPLE_STASH; ++q)
            if (np == q) { st_v[q] = v; st_k[q] = kbr; }
          ++np;
        }
      }
    }
    int block_total;
    const int excl = block_excl(np, sm, block_total);
    if (threadIdx.x < 32) {
      const int b = chain_exclusive(s.chain_t5, tile, block_total, threadIdx.x, epoch);
      if (threadIdx.x == 0) s_base = b;
    }
    __syncthreads();
    const int base = s_base;
    if (u < n && np) {
      int pos = base + excl;
      const float ku = s.t3_k[u];
      auto put = [&](int at, int v, float kbr) {
        const int4 cde = s.t3_abc[v];
        int* md = s.t5c_md + 5 * at;
        md[0] = abc.x; md[1] = abc.y; md[2] = abc.z; md[3] = cde.y; md[4] = cde.z;
        s.t5c_t3[at] = make_int2(u, v);
        float* cv = s.t5c_curv + 3 * at;
        cv[0] = ku; cv[1] = kbr; cv[2] = s.t3_k[v];
      };
      if (np <= TUPLE_STASH) {
#pragma unroll
        for (int q = 0; q < TUPLE_STASH; ++q)
          if (q < np && pos + q < cap) put(pos + q, st_v[q], st_k[q]);
      } else {
        for (int v = v0; v < v1; ++v) {
          const int d = s.t3_abc[v].y;
          const Pt D = make_pt(s.md_pos[d], s.md_modt[d] & 3);
          float kbr;
          if (!triplet_eval(B, C, D, kbr)) continue;
          if (pos < cap) put(pos, v, kbr);
          ++pos;
        }
      }
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
      const int total = base + block_total;
      s.cnt[LST_CNT_T5C] = min(total, cap);
      s.cnt[LST_CNT_RAW_T5C] = total;
      if (total > cap) atomicOr(reinterpret_cast<unsigned*>(s.cnt + CNT_STATUS), LST_ST_OVF_T5C);
    }
    __syncthreads();
  }
  LST_FOR_ITEMS(a, s.cnt[LST_CNT_MD] + 1) s.t3_start[a] = s.t3_off[s.ls_start[a]];      // (after the tiles: nobody here waits for it)
}

}  // namespace lst
