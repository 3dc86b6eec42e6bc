// oracle/lst_oracle.cpp -- TEST INFRASTRUCTURE ONLY (CPU oracle of the LST hot path).
//
// Plain, slow, single-threaded restatement of the chain the paper names
//   hits -> MD -> LS -> T3 -> T5 (+T5-DNN) -> track candidates   (Table 1 PAPER.md:45-60,
//   T5-DNN PAPER.md:62-68, :90)
// in the order and notation of SPEC.md (which freezes every cut the paper leaves out; each
// function below cites the SPEC.md section and the PAPER.md passage it follows).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code with paper_2403_13166_b200/ (the CUDA path)
// and neither includes the other; the product path never calls it.
//
// Precision: the north star fixes fp32 with a fixed operation order and no FMA contraction
// (compile with -ffp-contract=off, no fast-math).  The whole chain is a template on the real
// type so that tests can run a `double` instantiation of the same procedure as a pin.
//
// Parity status: the paper prints no cut value, object count or score for any input that can be
// constructed, so parity AGAINST THE PAPER is unpinned.  Against SPEC.md and
// mathematics every function below is pinned (tests/test_oracle_pins.py, tests/test_oracle_terms.py):
// brute-force enumeration, closed-form helices, textbook curvature cases, arcfac vs asin, an
// independent fp64 MLP, rotation / mirror / permutation invariance, cut-loosening monotonicity, and --
// term by term -- hand-derived accept / reject boundaries for every tolerance term of M2/M3, L1-L3,
// T1-T3, the anchor test and chi2, plus hand-built scenarios for run_chain's own assignments, the
// bridge indices and the TC used / free / tie rules.  The BUILD ORDER of every list (stable a0 sort,
// (m, i, j), CSR-row order, (l0, l1), (u, v)), the radius clamp and the sagitta cap of M3 are pinned by
// tests/test_oracle_order.py with numpy only.  tests/test_oracle_mutants.py shows that every entry of
// its MUTANTS table (single-line mutations of this file) fails at least one pin.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#include <algorithm>

namespace {

// ---------------------------------------------------------------- constants (SPEC.md 3.1)
constexpr float KAPPA_F = 0.0114f;        // GeV/cm = 0.3 * 3.8 T / 100
constexpr float C_HALF_F = 0.007125f;     // KAPPA / (2 PT_MIN), PT_MIN = 0.8 GeV
constexpr float C_MAX105_F = 0.0149625f;  // 1.05 KAPPA / PT_MIN
constexpr float C_TOL3_F = 0.00285f;      // 0.2 KAPPA / PT_MIN
constexpr float Z0_MAX_F = 15.0f;
constexpr float DT_F[2] = {0.01225f, 0.01102f};   // 3 sqrt2 sigma_t  (PS, 2S)
constexpr float DL_F[2] = {0.1299f, 4.330f};      // 3 sigma_l
constexpr float DL2_F[2] = {0.1837f, 6.124f};     // 3 sqrt2 sigma_l
constexpr int N_FEAT = 23, N_HID = 32, N_FEAT_MAX = 38;

// cut identifiers for the loosening factors (tests only; all 1.0 in normal use, and x*1.0 is exact)
enum { CUT_M2, CUT_M3, CUT_L1, CUT_L2, CUT_L3, CUT_T1, CUT_T2, CUT_T3, CUT_Q1, CUT_Q2, CUT_P5, CUT_P3, N_CUTS };

template <typename R> struct Loosen { R f[N_CUTS]; };

// ---------------------------------------------------------------- helpers (SPEC.md 3.2)
// arcfac(u) = asin(sqrt u)/sqrt u, 7-term Taylor in Horner form, separate mul/add.
template <typename R> inline R arcfac(R u) {
  R p = R(0.017352764f);
  p = R(0.022372159f) + u * p;
  p = R(0.030381944f) + u * p;
  p = R(0.044642857f) + u * p;
  p = R(0.075f) + u * p;
  p = R(0.16666667f) + u * p;
  p = R(1.0f) + u * p;
  return p;
}
template <typename R> inline R rabs(R v) { return std::fabs(v); }

// ---------------------------------------------------------------- objects
template <typename R> struct MD {
  int32_t hit_lo, hit_up;   // positions in the module-sorted hit store
  int32_t mod;
  R x, y, z, r;             // anchor = lower-sensor hit
  R c, w, f;                // signed curvature estimate, absolute tolerance, relative tolerance
  R dz, dr;                 // anchor long-direction tolerances
};
template <typename R> struct LS { int32_t a, b; R c; };
template <typename R> struct T3 { int32_t ls0, ls1; int32_t a, b, c; R k; };
template <typename R> struct T5C {
  int32_t t3in, t3out; int32_t md[5]; R cin, cbr, cout; float feat[N_FEAT_MAX]; float score; int8_t pass;
};
struct TC { int32_t type, pls, obj; };

// ---------------------------------------------------------------- step 1: MD (SPEC.md 4.1)
template <typename R>
inline bool md_eval(R x1, R y1, R z1, R x2, R y2, R z2, int subdet, int mtype, const Loosen<R>& lo,
                    R* c_out, R* w_out, R* f_out, R* r1_out) {
  const R r1 = std::sqrt(x1 * x1 + y1 * y1);
  const R r2 = std::sqrt(x2 * x2 + y2 * y2);
  const R dx = x2 - x1, dy = y2 - y1, dz = z2 - z1;
  const R drho = (x1 * dx + y1 * dy) / r1;
  const R dt = (x1 * dy - y1 * dx) / r1;
  const R S = std::fmin(R(1.0f), r2 * R(C_HALF_F));
  const R dtol = R(DT_F[mtype]);
  const R l2tol = R(DL2_F[mtype]);
  R c, w, f;
  if (subdet == 0) {
    if (!(drho > R(0.0f))) return false;                                             // M1
    const R L = std::sqrt(dt * dt + drho * drho);
    const R lhs2 = rabs(dz - drho * z1 / r1);
    const R rhs2 = drho * R(Z0_MAX_F) / r1 + l2tol;
    if (!(lhs2 <= rhs2 * lo.f[CUT_M2])) return false;                                // M2
    if (!(rabs(dt) <= (L * S + dtol) * lo.f[CUT_M3])) return false;                  // M3
    const R den = r2 * L;
    c = (R(-2.0f) * dt) / den;
    w = (R(2.0f) * dtol) / den;
    f = R(0.0f);
  } else {
    const R Ls = rabs(dz) * r1 / rabs(z1);
    if (!(rabs(drho - Ls) <= (R(0.15f) * Ls + l2tol) * lo.f[CUT_M2])) return false;  // M2
    if (!(rabs(dt) <= (R(1.3f) * Ls * S + dtol) * lo.f[CUT_M3])) return false;       // M3
    const R den = r2 * Ls;
    c = (R(-2.0f) * dt) / den;
    w = (R(2.0f) * dtol) / den;
    f = R(0.3f);
  }
  *c_out = c; *w_out = w; *f_out = f; *r1_out = r1;
  return true;
}

// ---------------------------------------------------------------- step 2: LS (SPEC.md 4.2)
template <typename R>
inline bool ls_eval(const MD<R>& A, const MD<R>& B, const Loosen<R>& lo, R* c_out) {
  const R dx = B.x - A.x, dy = B.y - A.y;
  const R d = std::sqrt(dx * dx + dy * dy);
  const R cr = A.x * dy - A.y * dx;
  const R c = (R(-2.0f) * cr) / ((A.r * B.r) * d);
  if (!(rabs(c) <= R(C_MAX105_F) * lo.f[CUT_L1])) return false;                      // L1
  const R ta = (A.r * c) * R(0.5f), tb = (B.r * c) * R(0.5f);
  const R sA = A.r * arcfac<R>(ta * ta);
  const R sB = B.r * arcfac<R>(tb * tb);
  const R lhs = rabs(A.z * sB - B.z * sA);
  R rhs = R(Z0_MAX_F) * rabs(sB - sA);
  rhs = rhs + A.dz * sB;
  rhs = rhs + B.dz * sA;
  rhs = rhs + A.dr * rabs(B.z);
  rhs = rhs + B.dr * rabs(A.z);
  if (!(lhs <= rhs * lo.f[CUT_L2])) return false;                                    // L2
  const R ac = rabs(c);
  if (!(rabs(A.c - c) <= (A.w + A.f * ac) * lo.f[CUT_L3])) return false;             // L3 (inner MD)
  if (!(rabs(B.c - c) <= (B.w + B.f * ac) * lo.f[CUT_L3])) return false;             // L3 (outer MD)
  *c_out = c;
  return true;
}

// 3-point (Menger) signed curvature and the r-z linearity test shared by T3 and the T5 bridge
// (SPEC.md 4.3; "radius of a simple circle fit").
template <typename R>
inline bool triplet_eval(const MD<R>& A, const MD<R>& B, const MD<R>& C, R f_curv, R f_rz, R* k_out) {
  const R abx = B.x - A.x, aby = B.y - A.y;
  const R acx = C.x - A.x, acy = C.y - A.y;
  const R bcx = C.x - B.x, bcy = C.y - B.y;
  const R dab = std::sqrt(abx * abx + aby * aby);
  const R dbc = std::sqrt(bcx * bcx + bcy * bcy);
  const R dac = std::sqrt(acx * acx + acy * acy);
  const R k = (R(-2.0f) * (abx * acy - aby * acx)) / ((dab * dbc) * dac);
  if (!(rabs(k) <= R(C_MAX105_F) * f_curv)) return false;                            // T1 / Q1
  const R tab = (dab * k) * R(0.5f), tbc = (dbc * k) * R(0.5f);
  const R sab = dab * arcfac<R>(tab * tab);
  const R sbc = dbc * arcfac<R>(tbc * tbc);
  const R zab = B.z - A.z, zbc = C.z - B.z;
  const R lhs = rabs(zab * sbc - zbc * sab);
  R rhs = (A.dz + B.dz) * sbc;
  rhs = rhs + (B.dz + C.dz) * sab;
  rhs = rhs + (A.dr + B.dr) * rabs(zbc);
  rhs = rhs + (B.dr + C.dr) * rabs(zab);
  rhs = rhs + R(0.05f) * (sab + sbc);
  if (!(lhs <= rhs * f_rz)) return false;                                            // T2 / Q2
  *k_out = k;
  return true;
}

// ---------------------------------------------------------------- step 3: T3 (SPEC.md 4.3)
template <typename R>
inline bool t3_eval(const MD<R>& A, const MD<R>& B, const MD<R>& C, R c_ab, R c_bc, const Loosen<R>& lo, R* k_out) {
  R k;
  if (!triplet_eval<R>(A, B, C, lo.f[CUT_T1], lo.f[CUT_T2], &k)) return false;
  if (!(rabs(c_ab - k) <= R(C_TOL3_F) * lo.f[CUT_T3])) return false;                 // T3
  if (!(rabs(c_bc - k) <= R(C_TOL3_F) * lo.f[CUT_T3])) return false;
  *k_out = k;
  return true;
}

// ---------------------------------------------------------------- step 4: features + DNN (SPEC.md 4.4, 4.5)
// Features and the MLP are fp32 in every instantiation (BASELINE.json configs[0]: "all data fp32").
inline float radius_feature(float c) {
  const float ac = std::fabs(c);
  const float rad = std::fmin(1.0f / ac, 1.0e5f);   // c = 0 -> +inf -> clamped
  return std::log10(rad);
}
inline void t5_features(const float* ax, const float* ay, const float* az, const float* ar,
                        float cin, float cbr, float cout, float* x) {
  for (int i = 0; i < 5; ++i) {
    x[4 * i + 0] = ar[i] * 0.01f;
    x[4 * i + 1] = az[i] * 0.01f;
    x[4 * i + 2] = std::asinh(az[i] / ar[i]);
    x[4 * i + 3] = std::atan2(ay[i], ax[i]);
  }
  x[20] = radius_feature(cin);
  x[21] = radius_feature(cbr);
  x[22] = radius_feature(cout);
}
// f3 (SPEC.md 4.9): the paper's 38 inputs -- 2 T3 x (pT, radius), 6 anchors (a, b, c, c, d, e) x (r, phi, z, eta, layer),
// T5 (pT, eta, phi), bridge radius
inline float pt_feature(float c) {
  const float ac = std::fabs(c);
  const float rad = std::fmin(1.0f / ac, 1.0e5f);
  return std::log10(KAPPA_F * rad);
}
inline void t5_features38(const float* ax, const float* ay, const float* az, const float* ar, const int* layer,
                          float cin, float cbr, float cout, float* x) {
  x[0] = pt_feature(cin); x[1] = radius_feature(cin); x[2] = pt_feature(cout); x[3] = radius_feature(cout);
  const int order[6] = {0, 1, 2, 2, 3, 4};
  for (int i = 0; i < 6; ++i) {
    const int q = order[i];
    x[4 + 5 * i + 0] = ar[q] * 0.01f;
    x[4 + 5 * i + 1] = std::atan2(ay[q], ax[q]);
    x[4 + 5 * i + 2] = az[q] * 0.01f;
    x[4 + 5 * i + 3] = std::asinh(az[q] / ar[q]);
    x[4 + 5 * i + 4] = float(layer[q]) * 0.1f;
  }
  const float c5 = 0.5f * (cin + cout);
  x[34] = pt_feature(c5);
  x[35] = std::asinh(az[0] / ar[0]);
  x[36] = std::atan2(ay[0], ax[0]);
  x[37] = radius_feature(cbr);
}
// "the DNN matrix multiplication is done through nested for-loops": acc = b[j];
// for i ascending: acc = acc + W[j][i] * x[i].  ReLU on every hidden layer, sigmoid output.  n_in inputs, n_hidden hidden
// layers of 32 (PAPER.md:68 has two; :78 scans one to four).
inline float mlp_forward(const float* w, const float* x, int n_in = N_FEAT, int n_hidden = 2) {
  float h[N_HID], g[N_HID];
  const float* W = w;
  const float* b = W + N_HID * n_in;
  for (int j = 0; j < N_HID; ++j) {
    float acc = b[j];
    for (int i = 0; i < n_in; ++i) acc = acc + W[j * n_in + i] * x[i];
    h[j] = acc > 0.0f ? acc : 0.0f;
  }
  const float* p = b + N_HID;
  for (int l = 1; l < n_hidden; ++l) {
    const float* Wl = p;
    const float* bl = Wl + N_HID * N_HID;
    for (int j = 0; j < N_HID; ++j) {
      float acc = bl[j];
      for (int i = 0; i < N_HID; ++i) acc = acc + Wl[j * N_HID + i] * h[i];
      g[j] = acc > 0.0f ? acc : 0.0f;
    }
    for (int j = 0; j < N_HID; ++j) h[j] = g[j];
    p = bl + N_HID;
  }
  const float* w3 = p;
  float y = w3[N_HID];
  for (int i = 0; i < N_HID; ++i) y = y + w3[i] * h[i];
  return 1.0f / (1.0f + std::exp(-y));
}

// ---------------------------------------------------------------- steps 5-8: pLS matching (SPEC.md 4.6)
template <typename R> struct PLS { R cx, cy, h, cot, sec, z0; };
template <typename R>
inline PLS<R> pls_derive(R px, R py, R pz, R z0, int q) {
  PLS<R> p;
  const R pt = std::sqrt(px * px + py * py);
  const R Rr = pt / R(KAPPA_F);
  const R qR = R(float(q)) * Rr;
  p.cx = (qR * py) / pt;
  p.cy = (-(qR * px)) / pt;
  p.h = R(0.5f) / Rr;
  p.cot = pz / pt;
  p.sec = std::sqrt(R(1.0f) + p.cot * p.cot);
  p.z0 = z0;
  return p;
}
// SPEC.md 4.6 [R20]: a pair only matches if its finished chi2 is a number below infinity.  On finite inputs every chi2 term is
// <= 1, so this never bites; a seed with pz = +-inf has dZ = inf, passes |zres| = inf <= dZ and would carry chi2 = NaN, for
// which argmin over (chi2, index) is undefined.
template <typename R>
inline bool chi2_is_a_number(R chi) { return chi < std::numeric_limits<R>::infinity(); }
// one anchor against one pLS helix; adds its two chi2 terms to *chi2 when it passes
template <typename R>
inline bool pls_anchor(const PLS<R>& p, const MD<R>& m, R loosen, R* chi2) {
  const R r2 = m.r * m.r;
  const R wv = m.x * p.cx + m.y * p.cy;
  const R e = (r2 - R(2.0f) * wv) * p.h;
  R dT = R(0.003f) * m.r;
  dT = dT + R(0.03f) * (r2 * p.h);
  dT = dT + R(0.02f);
  dT = dT * loosen;
  if (!(rabs(e) <= dT)) return false;
  const R t = m.r * p.h;
  const R s = m.r * arcfac<R>(t * t);
  const R zres = m.z - (p.z0 + s * p.cot);
  R dZ = m.dz + m.dr * rabs(p.cot);
  dZ = dZ + R(0.003f) * (s * p.sec);
  dZ = dZ + R(0.05f);
  dZ = dZ * loosen;
  if (!(rabs(zres) <= dZ)) return false;
  const R a = e / dT, b = zres / dZ;
  *chi2 = *chi2 + a * a;
  *chi2 = *chi2 + b * b;
  return true;
}

// ---------------------------------------------------------------- f1: duplicate cleaning (SPEC.md 4.7)
// rank key (type, q, row), smaller = better; X is a duplicate iff a better-ranked Y holds more than half of X's hits
inline bool better_rank(const TC& y, uint32_t qy, int32_t iy, const TC& x, uint32_t qx, int32_t ix) {
  if (y.type != x.type) return y.type < x.type;
  if (qy != qx) return qy < qx;
  return iy < ix;
}
inline void clean_duplicates(int32_t n, const TC* tc, const uint32_t* q, const int32_t* hits /*[n][10]*/, const int32_t* nh,
                             std::vector<int32_t>& keep) {
  keep.assign(n, 1);
  // Y can only hold more than half of X's hits if it holds at least one of them: list, per hit, the candidates that
  // contain it, and test X only against the candidates found under X's own hits (otherwise the plain all-pairs loop)
  int32_t max_hit = -1;
  for (int32_t i = 0; i < n; ++i) for (int a = 0; a < nh[i]; ++a) max_hit = std::max(max_hit, hits[10 * i + a]);
  std::vector<std::vector<int32_t>> holders(size_t(max_hit + 1));
  for (int32_t i = 0; i < n; ++i) if (tc[i].type <= 2) for (int a = 0; a < nh[i]; ++a) holders[hits[10 * i + a]].push_back(i);
  for (int32_t x = 0; x < n; ++x) {
    if (tc[x].type > 2) continue;                       // pLS candidates carry no outer-tracker hits
    for (int a0 = 0; a0 < nh[x] && keep[x]; ++a0) {
      for (int32_t y : holders[hits[10 * x + a0]]) {
        if (y == x || !better_rank(tc[y], q[y], y, tc[x], q[x], x)) continue;
        int shared = 0;
        for (int a = 0; a < nh[x]; ++a) {               // slots of X whose hit occurs anywhere in Y
          bool in_y = false;
          for (int b = 0; b < nh[y]; ++b) in_y = in_y || hits[10 * y + b] == hits[10 * x + a];
          shared += in_y;
        }
        if (2 * shared > nh[x]) keep[x] = 0;
      }
    }
  }
}

// ---------------------------------------------------------------- the chain
template <typename R> struct Result {
  uint32_t flags = 0;                 // bit 0: a hit key was out of range (hit dropped)
  std::vector<int32_t> hit_orig;      // sorted position -> original hit index
  std::vector<int32_t> sensor_start;  // [2M+1]
  std::vector<MD<R>> md;
  std::vector<int32_t> md_start;      // [M+1] MDs of module m
  std::vector<LS<R>> ls;
  std::vector<int32_t> ls_start;      // [N_md+1] LSs whose inner MD is a
  std::vector<T3<R>> t3;
  std::vector<int32_t> t3_start;      // [N_md+1] T3s whose inner MD is a
  std::vector<T5C<R>> t5c;
  std::vector<int32_t> t5;            // candidate indices passing the DNN
  std::vector<TC> tc;
  std::vector<int32_t> best5_pls;     // per T5: best matching pLS or -1
  std::vector<float> chi5;            // per T5: chi2 of that match
  std::vector<float> chi3;            // per T3: chi2 of its best free-seed match (0 if none)
  std::vector<int32_t> tc_keep;       // per TC row: 1 = kept by the duplicate cleaning (SPEC.md 4.7)
  std::vector<int32_t> tc_hits;       // per TC row: its 10 ORIGINAL hit indices (-1 padded), the tuple the cleaning compares
  std::vector<int32_t> tc_q;          // per TC row: chi2 bit pattern that enters its rank key
  std::vector<TC> tcc;                // cleaned TC list
  int64_t n_md_pairs = 0, n_ls_pairs = 0, n_t3_pairs = 0, n_t5_pairs = 0, n_match5 = 0, n_match3 = 0;
};

template <typename R>
Result<R>* run_chain(int32_t M, const uint8_t* subdet, const uint8_t* mtype, const int32_t* rowptr,
                     const int32_t* col, const float* weights, int32_t n_hits, const float* hx,
                     const float* hy, const float* hz, const uint32_t* key, int32_t n_pls,
                     const float* ppx, const float* ppy, const float* ppz, const float* pz0,
                     const int8_t* pq, const int8_t* t5_override, int32_t n_override,
                     const float* loosen, int32_t last_stage, int32_t n_feat = N_FEAT, int32_t n_hidden = 2,
                     const uint8_t* layer = nullptr) {
  Result<R>* res = new Result<R>();
  Loosen<R> lo;
  for (int i = 0; i < N_CUTS; ++i) lo.f[i] = loosen ? R(loosen[i]) : R(1.0f);

  // ---- a0: stable counting sort of hits by sensor key = 2*module + isUpper (SPEC.md 4.0)
  const int32_t S = 2 * M;
  res->sensor_start.assign(S + 1, 0);
  for (int32_t i = 0; i < n_hits; ++i) {
    if (key[i] >= uint32_t(S)) { res->flags |= 1u; continue; }
    res->sensor_start[key[i] + 1]++;
  }
  for (int32_t s = 0; s < S; ++s) res->sensor_start[s + 1] += res->sensor_start[s];
  res->hit_orig.assign(res->sensor_start[S], 0);
  {
    std::vector<int32_t> cur(res->sensor_start.begin(), res->sensor_start.end() - 1);
    for (int32_t i = 0; i < n_hits; ++i) {
      if (key[i] >= uint32_t(S)) continue;
      res->hit_orig[cur[key[i]]++] = i;
    }
  }
  const std::vector<int32_t>& ho = res->hit_orig;
  const std::vector<int32_t>& ss = res->sensor_start;
  if (last_stage < 1) return res;

  // ---- a1: MD -- for module -> for lower hit -> for upper hit
  res->md_start.assign(M + 1, 0);
  for (int32_t m = 0; m < M; ++m) {
    res->md_start[m] = int32_t(res->md.size());
    for (int32_t i = ss[2 * m]; i < ss[2 * m + 1]; ++i) {
      for (int32_t j = ss[2 * m + 1]; j < ss[2 * m + 2]; ++j) {
        res->n_md_pairs++;
        const int32_t oi = ho[i], oj = ho[j];
        MD<R> d;
        if (!md_eval<R>(R(hx[oi]), R(hy[oi]), R(hz[oi]), R(hx[oj]), R(hy[oj]), R(hz[oj]), subdet[m],
                        mtype[m], lo, &d.c, &d.w, &d.f, &d.r))
          continue;
        d.hit_lo = i; d.hit_up = j; d.mod = m;
        d.x = R(hx[oi]); d.y = R(hy[oi]); d.z = R(hz[oi]);
        d.dz = subdet[m] == 0 ? R(DL_F[mtype[m]]) : R(0.0f);
        d.dr = subdet[m] == 0 ? R(0.0f) : R(DL_F[mtype[m]]);
        res->md.push_back(d);
      }
    }
  }
  res->md_start[M] = int32_t(res->md.size());
  const int32_t n_md = int32_t(res->md.size());
  if (last_stage < 2) return res;

  // ---- a2: LS -- for MD a -> for m' in CSR row of module(a) -> for MD b in m'
  res->ls_start.assign(n_md + 1, 0);
  for (int32_t a = 0; a < n_md; ++a) {
    res->ls_start[a] = int32_t(res->ls.size());
    const int32_t m = res->md[a].mod;
    for (int32_t e = rowptr[m]; e < rowptr[m + 1]; ++e) {
      const int32_t m2 = col[e];
      for (int32_t b = res->md_start[m2]; b < res->md_start[m2 + 1]; ++b) {
        res->n_ls_pairs++;
        R c;
        if (!ls_eval<R>(res->md[a], res->md[b], lo, &c)) continue;
        res->ls.push_back(LS<R>{a, b, c});
      }
    }
  }
  res->ls_start[n_md] = int32_t(res->ls.size());
  const int32_t n_ls = int32_t(res->ls.size());
  if (last_stage < 3) return res;

  // ---- a3: T3 -- for LS (a,b) -> for LS (b,c)
  res->t3_start.assign(n_md + 1, 0);
  {
    int32_t a_prev = 0;
    for (int32_t l0 = 0; l0 < n_ls; ++l0) {
      const LS<R>& s0 = res->ls[l0];
      while (a_prev <= s0.a) res->t3_start[a_prev++] = int32_t(res->t3.size());
      for (int32_t l1 = res->ls_start[s0.b]; l1 < res->ls_start[s0.b + 1]; ++l1) {
        const LS<R>& s1 = res->ls[l1];
        res->n_t3_pairs++;
        R k;
        if (!t3_eval<R>(res->md[s0.a], res->md[s0.b], res->md[s1.b], s0.c, s1.c, lo, &k)) continue;
        res->t3.push_back(T3<R>{l0, l1, s0.a, s0.b, s1.b, k});
      }
    }
    while (a_prev <= n_md) res->t3_start[a_prev++] = int32_t(res->t3.size());
  }
  const int32_t n_t3 = int32_t(res->t3.size());
  if (last_stage < 4) return res;

  // ---- a4 + a5: T5 candidates -- for T3 (a,b,c) -> for T3 (c,d,e); bridge (b,c,d); DNN per candidate
  for (int32_t i0 = 0; i0 < n_t3; ++i0) {
    const T3<R>& u = res->t3[i0];
    for (int32_t i1 = res->t3_start[u.c]; i1 < res->t3_start[u.c + 1]; ++i1) {
      const T3<R>& v = res->t3[i1];
      res->n_t5_pairs++;
      R kbr;
      if (!triplet_eval<R>(res->md[u.b], res->md[u.c], res->md[v.b], lo.f[CUT_Q1], lo.f[CUT_Q2], &kbr)) continue;
      T5C<R> t;
      t.t3in = i0; t.t3out = i1;
      t.md[0] = u.a; t.md[1] = u.b; t.md[2] = u.c; t.md[3] = v.b; t.md[4] = v.c;
      t.cin = u.k; t.cbr = kbr; t.cout = v.k;
      float ax[5], ay[5], az[5], ar[5];
      for (int q = 0; q < 5; ++q) {
        const MD<R>& d = res->md[t.md[q]];
        ax[q] = float(d.x); ay[q] = float(d.y); az[q] = float(d.z); ar[q] = float(d.r);
      }
      for (int q = 0; q < N_FEAT_MAX; ++q) t.feat[q] = 0.0f;
      if (n_feat == N_FEAT_MAX) {
        int lay[5];
        for (int q = 0; q < 5; ++q) lay[q] = layer ? int(layer[res->md[t.md[q]].mod]) : 0;
        t5_features38(ax, ay, az, ar, lay, float(t.cin), float(t.cbr), float(t.cout), t.feat);
      } else {
        t5_features(ax, ay, az, ar, float(t.cin), float(t.cbr), float(t.cout), t.feat);
      }
      t.score = mlp_forward(weights, t.feat, n_feat, n_hidden);
      t.pass = t.score > 0.5f ? 1 : 0;
      const int32_t ci = int32_t(res->t5c.size());
      if (t5_override && ci < n_override && t5_override[ci] >= 0) t.pass = t5_override[ci];
      if (t.pass) res->t5.push_back(ci);
      res->t5c.push_back(t);
    }
  }
  const int32_t n_t5 = int32_t(res->t5.size());
  if (last_stage < 5) return res;

  // ---- a6: track candidates (Table 1 steps 5-8)
  std::vector<PLS<R>> pls(n_pls);
  for (int32_t p = 0; p < n_pls; ++p) pls[p] = pls_derive<R>(R(ppx[p]), R(ppy[p]), R(ppz[p]), R(pz0[p]), pq[p]);
  // best5(t) = argmin_p (chi2, p) over matching p
  res->best5_pls.assign(n_t5, -1);
  res->chi5.assign(n_t5, 0.0f);
  std::vector<R> chi5(n_t5, R(0));
  for (int32_t t = 0; t < n_t5; ++t) {
    const T5C<R>& q5 = res->t5c[res->t5[t]];
    for (int32_t p = 0; p < n_pls; ++p) {
      R chi = R(0.0f);
      bool ok = true;
      for (int q = 0; q < 5 && ok; ++q) ok = pls_anchor<R>(pls[p], res->md[q5.md[q]], lo.f[CUT_P5], &chi);
      if (!ok || !chi2_is_a_number<R>(chi)) continue;   // T5 match
      res->n_match5++;
      if (res->best5_pls[t] < 0 || chi < chi5[t]) { res->best5_pls[t] = p; chi5[t] = chi; }
    }
    res->chi5[t] = float(chi5[t]);
  }
  // win5(p) = argmin_t (chi2, t) over {t : best5(t) = p}
  std::vector<int32_t> win5(n_pls, -1);
  for (int32_t t = 0; t < n_t5; ++t) {
    const int32_t p = res->best5_pls[t];
    if (p < 0) continue;
    if (win5[p] < 0 || chi5[t] < chi5[win5[p]]) win5[p] = t;
  }
  // eligible T3s: not contained in the five MDs of any pT5
  std::vector<uint8_t> t3_used(n_t3, 0);
  for (int32_t x = 0; x < n_t3; ++x) {
    const T3<R>& u = res->t3[x];
    for (int32_t p = 0; p < n_pls && !t3_used[x]; ++p) {
      if (win5[p] < 0) continue;
      const int32_t* m5 = res->t5c[res->t5[win5[p]]].md;
      int found = 0;
      for (int q = 0; q < 5; ++q) found += (m5[q] == u.a) + (m5[q] == u.b) + (m5[q] == u.c);
      if (found == 3) t3_used[x] = 1;
    }
  }
  // best3(x) over free pLS, win3(p) over eligible T3
  std::vector<int32_t> best3(n_t3, -1), win3(n_pls, -1);
  std::vector<R> chi3(n_t3, R(0));
  for (int32_t x = 0; x < n_t3; ++x) {
    if (t3_used[x]) continue;
    const T3<R>& u = res->t3[x];
    const int32_t mm[3] = {u.a, u.b, u.c};
    for (int32_t p = 0; p < n_pls; ++p) {
      if (win5[p] >= 0) continue;
      R chi = R(0.0f);
      bool ok = true;
      for (int q = 0; q < 3 && ok; ++q) ok = pls_anchor<R>(pls[p], res->md[mm[q]], lo.f[CUT_P3], &chi);
      if (!ok || !chi2_is_a_number<R>(chi)) continue;   // T3 match
      res->n_match3++;
      if (best3[x] < 0 || chi < chi3[x]) { best3[x] = p; chi3[x] = chi; }
    }
  }
  for (int32_t x = 0; x < n_t3; ++x) {
    const int32_t p = best3[x];
    if (p < 0) continue;
    if (win3[p] < 0 || chi3[x] < chi3[win3[p]]) win3[p] = x;
  }
  res->chi3.assign(n_t3, 0.0f);
  for (int32_t x = 0; x < n_t3; ++x) res->chi3[x] = float(chi3[x]);
  // emit: pT5 (by p), T5 (by t), pT3 (by p), pLS (by p) -- mutually exclusive
  for (int32_t p = 0; p < n_pls; ++p) if (win5[p] >= 0) res->tc.push_back(TC{0, p, win5[p]});
  for (int32_t t = 0; t < n_t5; ++t) if (res->best5_pls[t] < 0) res->tc.push_back(TC{1, -1, t});
  for (int32_t p = 0; p < n_pls; ++p) if (win5[p] < 0 && win3[p] >= 0) res->tc.push_back(TC{2, p, win3[p]});
  for (int32_t p = 0; p < n_pls; ++p) if (win5[p] < 0 && win3[p] < 0) res->tc.push_back(TC{3, p, -1});
  if (last_stage < 6) return res;

  // ---- f1: duplicate cleaning (SPEC.md 4.7)
  {
    const int32_t n_tc = int32_t(res->tc.size());
    std::vector<int32_t> hits(size_t(n_tc) * 10, -1), nh(n_tc, 0);
    std::vector<uint32_t> q(n_tc, 0u);
    for (int32_t i = 0; i < n_tc; ++i) {
      const TC& c = res->tc[i];
      int32_t mds[5], nm = 0;
      if (c.type <= 1) { const int32_t* m5 = res->t5c[res->t5[c.obj]].md; for (int k = 0; k < 5; ++k) mds[k] = m5[k]; nm = 5; }
      else if (c.type == 2) { const T3<R>& u = res->t3[c.obj]; mds[0] = u.a; mds[1] = u.b; mds[2] = u.c; nm = 3; }
      for (int k = 0; k < nm; ++k) { hits[10 * i + 2 * k] = ho[res->md[mds[k]].hit_lo]; hits[10 * i + 2 * k + 1] = ho[res->md[mds[k]].hit_up]; }
      nh[i] = 2 * nm;
      float chi = 0.0f;
      if (c.type == 0) chi = res->chi5[c.obj];
      if (c.type == 2) chi = res->chi3[c.obj];
      std::memcpy(&q[i], &chi, 4);
    }
    clean_duplicates(n_tc, res->tc.data(), q.data(), hits.data(), nh.data(), res->tc_keep);
    res->tc_hits = hits;
    res->tc_q.assign(q.begin(), q.end());
    for (int32_t i = 0; i < n_tc; ++i) if (res->tc_keep[i]) res->tcc.push_back(res->tc[i]);
  }
  return res;
}

struct Handle { int is_double; void* p; };

template <typename R> int64_t count_of(const Result<R>* r, int what) {
  switch (what) {
    case 0: return int64_t(r->hit_orig.size());
    case 1: return int64_t(r->md.size());
    case 2: return int64_t(r->ls.size());
    case 3: return int64_t(r->t3.size());
    case 4: return int64_t(r->t5c.size());
    case 5: return int64_t(r->t5.size());
    case 6: return int64_t(r->tc.size());
    case 8: return int64_t(r->tcc.size());
    case 10: return r->n_md_pairs;
    case 11: return r->n_ls_pairs;
    case 12: return r->n_t3_pairs;
    case 13: return r->n_t5_pairs;
    case 14: return r->n_match5;
    case 15: return r->n_match3;
    case 20: return int64_t(r->flags);
    case 21: return int64_t(r->sensor_start.size());
    case 22: return int64_t(r->ls_start.size());
  }
  return -1;
}

// Copy-out: integer tables as int32 [n][k], real payloads as double [n][k] (exact for fp32).
template <typename R> void copy_int(const Result<R>* r, int what, int32_t* o) {
  const std::vector<int32_t>& ho = r->hit_orig;
  switch (what) {
    case 0: for (size_t i = 0; i < ho.size(); ++i) o[i] = ho[i]; break;
    case 1: for (size_t i = 0; i < r->md.size(); ++i) {                     // [n][3] orig hit lo, up, module
        o[3 * i] = ho[r->md[i].hit_lo]; o[3 * i + 1] = ho[r->md[i].hit_up]; o[3 * i + 2] = r->md[i].mod; } break;
    case 2: for (size_t i = 0; i < r->ls.size(); ++i) { o[2 * i] = r->ls[i].a; o[2 * i + 1] = r->ls[i].b; } break;
    case 3: for (size_t i = 0; i < r->t3.size(); ++i) {                     // [n][5] md a,b,c, ls0, ls1
        const T3<R>& t = r->t3[i]; o[5 * i] = t.a; o[5 * i + 1] = t.b; o[5 * i + 2] = t.c; o[5 * i + 3] = t.ls0; o[5 * i + 4] = t.ls1; } break;
    case 4: for (size_t i = 0; i < r->t5c.size(); ++i) {                    // [n][8] md[5], t3in, t3out, pass
        const T5C<R>& t = r->t5c[i]; for (int q = 0; q < 5; ++q) o[8 * i + q] = t.md[q];
        o[8 * i + 5] = t.t3in; o[8 * i + 6] = t.t3out; o[8 * i + 7] = t.pass; } break;
    case 5: for (size_t i = 0; i < r->t5.size(); ++i) o[i] = r->t5[i]; break;
    case 6: for (size_t i = 0; i < r->tc.size(); ++i) { o[3 * i] = r->tc[i].type; o[3 * i + 1] = r->tc[i].pls; o[3 * i + 2] = r->tc[i].obj; } break;
    case 7: for (size_t i = 0; i < r->best5_pls.size(); ++i) o[i] = r->best5_pls[i]; break;
    case 8: for (size_t i = 0; i < r->tcc.size(); ++i) { o[3 * i] = r->tcc[i].type; o[3 * i + 1] = r->tcc[i].pls; o[3 * i + 2] = r->tcc[i].obj; } break;
    case 9: for (size_t i = 0; i < r->tc_keep.size(); ++i) o[i] = r->tc_keep[i]; break;
    case 10: for (size_t i = 0; i < r->tc_hits.size(); ++i) o[i] = r->tc_hits[i]; break;
    case 11: for (size_t i = 0; i < r->tc_q.size(); ++i) o[i] = r->tc_q[i]; break;
    case 12: for (size_t i = 0; i < r->ls_start.size(); ++i) o[i] = r->ls_start[i]; break;       // f4: CSR rowptr of the MD/LS graph
    case 21: for (size_t i = 0; i < r->sensor_start.size(); ++i) o[i] = r->sensor_start[i]; break;
  }
}
template <typename R> void copy_real(const Result<R>* r, int what, double* o) {
  switch (what) {
    case 1: for (size_t i = 0; i < r->md.size(); ++i) {                     // [n][6] c, w, x, y, z, r
        const MD<R>& d = r->md[i]; double* q = o + 6 * i;
        q[0] = double(d.c); q[1] = double(d.w); q[2] = double(d.x); q[3] = double(d.y); q[4] = double(d.z); q[5] = double(d.r); } break;
    case 2: for (size_t i = 0; i < r->ls.size(); ++i) o[i] = double(r->ls[i].c); break;
    case 3: for (size_t i = 0; i < r->t3.size(); ++i) o[i] = double(r->t3[i].k); break;
    case 4: for (size_t i = 0; i < r->t5c.size(); ++i) {                    // [n][42] cin, cbr, cout, score, feat[38] (unused = 0)
        const T5C<R>& t = r->t5c[i]; double* q = o + 42 * i;
        q[0] = double(t.cin); q[1] = double(t.cbr); q[2] = double(t.cout); q[3] = double(t.score);
        for (int f = 0; f < N_FEAT_MAX; ++f) q[4 + f] = double(t.feat[f]); } break;
    case 7: for (size_t i = 0; i < r->chi5.size(); ++i) o[i] = double(r->chi5[i]); break;
    case 9: for (size_t i = 0; i < r->chi3.size(); ++i) o[i] = double(r->chi3[i]); break;
    case 12: for (size_t i = 0; i < r->md.size(); ++i) {                    // f4 (SPEC.md 4.8): node features [n][8], fp32 arithmetic
        const MD<R>& d = r->md[i]; double* q = o + 8 * i;
        const float x = float(d.x), y = float(d.y), z = float(d.z), rr = float(d.r);
        q[0] = x; q[1] = y; q[2] = z; q[3] = rr; q[4] = std::atan2(y, x); q[5] = std::asinh(z / rr); q[6] = double(float(d.c)); q[7] = double(float(d.w)); } break;
  }
}

}  // namespace

extern "C" {

void* lst_oracle_run(int32_t n_modules, const uint8_t* subdet, const uint8_t* mtype, const int32_t* rowptr,
                     const int32_t* col, const float* weights, int32_t n_hits, const float* x, const float* y,
                     const float* z, const uint32_t* key, int32_t n_pls, const float* px, const float* py,
                     const float* pz, const float* z0, const int8_t* q, const int8_t* t5_override,
                     int32_t n_override, const float* loosen, int32_t use_double, int32_t last_stage,
                     int32_t n_feat, int32_t n_hidden, const uint8_t* layer) {
  Handle* h = new Handle();
  h->is_double = use_double;
  if (use_double)
    h->p = run_chain<double>(n_modules, subdet, mtype, rowptr, col, weights, n_hits, x, y, z, key, n_pls, px, py,
                             pz, z0, q, t5_override, n_override, loosen, last_stage, n_feat, n_hidden, layer);
  else
    h->p = run_chain<float>(n_modules, subdet, mtype, rowptr, col, weights, n_hits, x, y, z, key, n_pls, px, py,
                            pz, z0, q, t5_override, n_override, loosen, last_stage, n_feat, n_hidden, layer);
  return h;
}
int64_t lst_oracle_count(void* hv, int32_t what) {
  Handle* h = static_cast<Handle*>(hv);
  return h->is_double ? count_of(static_cast<Result<double>*>(h->p), what) : count_of(static_cast<Result<float>*>(h->p), what);
}
void lst_oracle_copy_int(void* hv, int32_t what, int32_t* out) {
  Handle* h = static_cast<Handle*>(hv);
  if (h->is_double) copy_int(static_cast<Result<double>*>(h->p), what, out);
  else copy_int(static_cast<Result<float>*>(h->p), what, out);
}
void lst_oracle_copy_real(void* hv, int32_t what, double* out) {
  Handle* h = static_cast<Handle*>(hv);
  if (h->is_double) copy_real(static_cast<Result<double>*>(h->p), what, out);
  else copy_real(static_cast<Result<float>*>(h->p), what, out);
}
void lst_oracle_free(void* hv) {
  Handle* h = static_cast<Handle*>(hv);
  if (h->is_double) delete static_cast<Result<double>*>(h->p);
  else delete static_cast<Result<float>*>(h->p);
  delete h;
}

// ---- single-predicate entry points (brute-force and closed-form pins call these directly)
static MD<float> mk_md(const float* a) {   // a = x, y, z, r, c, w, f, dz, dr
  MD<float> m; m.hit_lo = m.hit_up = m.mod = 0;
  m.x = a[0]; m.y = a[1]; m.z = a[2]; m.r = a[3]; m.c = a[4]; m.w = a[5]; m.f = a[6]; m.dz = a[7]; m.dr = a[8];
  return m;
}
static Loosen<float> unit_loosen() { Loosen<float> l; for (int i = 0; i < N_CUTS; ++i) l.f[i] = 1.0f; return l; }

// out = c, w, f, r1, dz, dr
int32_t lst_oracle_md_eval(const float* h1, const float* h2, int32_t subdet, int32_t mtype, float* out) {
  float c, w, f, r1;
  if (!md_eval<float>(h1[0], h1[1], h1[2], h2[0], h2[1], h2[2], subdet, mtype, unit_loosen(), &c, &w, &f, &r1)) return 0;
  out[0] = c; out[1] = w; out[2] = f; out[3] = r1;
  out[4] = subdet == 0 ? DL_F[mtype] : 0.0f; out[5] = subdet == 0 ? 0.0f : DL_F[mtype];
  return 1;
}
int32_t lst_oracle_ls_eval(const float* a, const float* b, float* c_out) {
  return ls_eval<float>(mk_md(a), mk_md(b), unit_loosen(), c_out) ? 1 : 0;
}
int32_t lst_oracle_t3_eval(const float* a, const float* b, const float* c, float c_ab, float c_bc, float* k_out) {
  return t3_eval<float>(mk_md(a), mk_md(b), mk_md(c), c_ab, c_bc, unit_loosen(), k_out) ? 1 : 0;
}
int32_t lst_oracle_bridge_eval(const float* a, const float* b, const float* c, float* k_out) {
  return triplet_eval<float>(mk_md(a), mk_md(b), mk_md(c), 1.0f, 1.0f, k_out) ? 1 : 0;
}
// anchors: n rows of 9 floats (mk_md layout); returns 1 + chi2 when every anchor passes
int32_t lst_oracle_pls_match(const float* pls5, int32_t q, const float* anchors, int32_t n, float* chi2_out) {
  PLS<float> p = pls_derive<float>(pls5[0], pls5[1], pls5[2], pls5[3], q);
  float chi = 0.0f;
  for (int i = 0; i < n; ++i)
    if (!pls_anchor<float>(p, mk_md(anchors + 9 * i), 1.0f, &chi)) return 0;
  if (!chi2_is_a_number<float>(chi)) return 0;
  *chi2_out = chi;
  return 1;
}
// residuals of one anchor in double (closed-form pin: exactly 0 on the generating helix)
void lst_oracle_pls_residual(const double* pls5, int32_t q, const double* xyz, double* out) {
  PLS<double> p = pls_derive<double>(pls5[0], pls5[1], pls5[2], pls5[3], q);
  const double r = std::sqrt(xyz[0] * xyz[0] + xyz[1] * xyz[1]);
  const double e = (r * r - 2.0 * (xyz[0] * p.cx + xyz[1] * p.cy)) * p.h;
  const double t = r * p.h;
  const double s = r * arcfac<double>(t * t);
  out[0] = e; out[1] = xyz[2] - (p.z0 + s * p.cot); out[2] = s;
}
// duplicate cleaning on hand-made candidates: types[n], q[n] (chi2 bit patterns), hits[n][10] (-1 padded), nh[n] -> keep[n]
void lst_oracle_tc_clean(int32_t n, const int32_t* types, const uint32_t* q, const int32_t* hits, const int32_t* nh, int32_t* keep_out) {
  std::vector<TC> tc(n);
  for (int i = 0; i < n; ++i) tc[i] = TC{types[i], -1, -1};
  std::vector<int32_t> keep;
  clean_duplicates(n, tc.data(), q, hits, nh, keep);
  for (int i = 0; i < n; ++i) keep_out[i] = keep[i];
}
float lst_oracle_arcfac(float u) { return arcfac<float>(u); }
double lst_oracle_arcfac_f64(double u) { return arcfac<double>(u); }
void lst_oracle_features(const float* ax, const float* ay, const float* az, const float* ar, float cin, float cbr,
                         float cout, float* x23) { t5_features(ax, ay, az, ar, cin, cbr, cout, x23); }
float lst_oracle_mlp(const float* weights, const float* x23) { return mlp_forward(weights, x23); }
float lst_oracle_mlp_n(const float* weights, const float* x, int32_t n_in, int32_t n_hidden) { return mlp_forward(weights, x, n_in, n_hidden); }
void lst_oracle_features38(const float* ax, const float* ay, const float* az, const float* ar, const int32_t* layer, float cin,
                           float cbr, float cout, float* x38) { t5_features38(ax, ay, az, ar, layer, cin, cbr, cout, x38); }

}  // extern "C"
