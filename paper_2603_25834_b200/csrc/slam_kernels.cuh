// Hand-written sm_100a kernels of the batched fixed-lag SE(2) smoother: device phases of the fused step
// kernel (slam_api.cu).  A TEAM of 32/64/128 threads owns one environment; everything between loading
// and storing its record lives in shared memory.
//
// Hot path: per environment and per step
//   S0 push        dead-reckoned guess + factor bookkeeping
//   S1 linearise   residuals + SE(2) Jacobians of every live factor              (eq. (5))
//   S2 assemble    H = Lambda + sum J'Omega J, b, in shared memory, envelope (skyline) storage in 4x4 tiles
//   S3 factor      left-looking envelope Cholesky by 4-column blocks: row pairs per thread, 128-bit loads,
//                  compact active-pair lists, K-split; the rhs rides along as an extra row (forward solve
//                  for free); blocked back substitution; additive update
//   S4 covariance  trailing 6x6 of L -> Sigma_t (global coords), ln det      (eq. (6))
//   S5 marginalise re-anchor + Schur complement of the oldest pose on the prior's support
//
// Elimination order of the window variables (scalar offsets), chosen per environment:
//   [ passive landmarks | e_1 .. e_{W-2} (chain, 3 each) | observed landmarks | pad | newest pose e_{c-1} (3) | anchor a (3) ]
// (pad = 0..3 dummy identity rows so that the dimension np is a multiple of 4) so that the covariance
// read-out needs only the trailing 6x6 of L.  Poses are robot-centric (anchor frame), landmarks global
// (reading R17b).  Row np of the envelope storage is the right-hand side b (row index np+1 aliases it).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "slam_layout.h"

namespace slamk {

enum { F_PUSH = 1, F_OBS0 = 2, F_COV = 4, F_MARG = 8, F_COPYCOV = 16 };
enum { ENV_NOT_PD = 1, ENV_NONFINITE = 2, ENV_ILLCOND = 8 };  // ILLCOND is internal: never stored in the status word

struct StepIO {
  const float* odom; const int32_t* lc_back; const float* lc_meas; const uint32_t* rb_mask; const float* rb_meas;
  float* cov; float* logdet; float* dopt; float* last_pose;
  float* cov_cache;  // [10][N]: 9 covariance entries + logdet
  // NEXT-1: unary absolute-pose factor for the pose this push appends (NULL: none)
  const float* un_pose; const float* un_info; const int32_t* un_valid;
};

struct WS {  // per-team views into shared memory
  float* st; int* lct; float* cs; uint32_t* rbm;
  uint32_t* rbf;   // per matrix row: offset such that H(i,j) = H[rbase + j] (16 bit) | first column / 4 (bits 16..)
  uint32_t* sup;   // per prior-support scalar: elimination offset (9 bit) | state index (9 bit) | angle flag (bit 18)
  float* sds;      // prior displacement, anchor-frame landmarks; scratch of the symbolic phase
  uint32_t* amask; // tables of the factorisation (pool)
  float* H;        // envelope of H + rhs rows (pool)
};

__device__ __forceinline__ WS make_ws(const Layout& ly, float* base) {
  WS w;
  w.st = base + ly.s_st;
  w.lct = (int*)(base + ly.s_lct); w.cs = base + ly.s_cs; w.rbm = (uint32_t*)(base + ly.s_rbm);
  w.rbf = (uint32_t*)(base + ly.s_rbf); w.sup = (uint32_t*)(base + ly.s_sup); w.sds = base + ly.s_sds;
  w.amask = nullptr; w.H = nullptr;  // set once the environment has its share of the CTA pool (slam_step_kernel)
  return w;
}
__device__ __forceinline__ int rb_of(const WS& w, int i) { return (int)(w.rbf[i] & 0xffffu); }
__device__ __forceinline__ int first_of(const WS& w, int i) { return (int)(w.rbf[i] >> 16) << 2; }
__device__ __forceinline__ int sup_off(uint32_t e) { return (int)(e & 0x1ffu); }
__device__ __forceinline__ int sup_idx(uint32_t e) { return (int)((e >> 9) & 0x1ffu); }
__device__ __forceinline__ bool sup_angle(uint32_t e) { return (e >> 18) & 1u; }

// ------------------------------------------------------------------ small helpers
#define FULLMASK 0xffffffffu
#ifndef SLAM_KUNROLL
#define SLAM_KUNROLL 1   // unroll factor of the factorisation's dot-product loop
#endif
#ifndef SLAM_KSPLIT_MIN
#define SLAM_KSPLIT_MIN 32  // shortest dot product (columns) for which lanes split the range
#endif

__device__ __forceinline__ float wrapf(float x) {  // to [-pi, pi], 2*pi split hi/lo
  const float k = rintf(x * 0.15915494309189535f);
  x = fmaf(-k, 6.2831854820251465f, x);
  return fmaf(-k, -1.7484555e-7f, x);
}
// sin and cos for |x| up to a few pi (every angle here is wrapped): quadrant reduction with a hi/lo
// split of pi/2 and the classic single-precision minimax kernels (Cephes sinf/cosf coefficients),
// ~1e-7 absolute.  Replaces sincosf, whose inlined large-argument slow path bloats the kernel: the
// step kernel is instruction-fetch bound, so code size is a first-order cost.
__device__ __forceinline__ void sincos_pi(float x, float* sn, float* cn) {
  const float k = rintf(x * 0.63661977236758134f);
  float r = fmaf(-k, 1.5707963705062866f, x);
  r = fmaf(-k, -4.3711388286737929e-8f, r);
  const float z = r * r;
  const float sp = fmaf(fmaf(fmaf(-1.9515295891e-4f, z, 8.3321608736e-3f), z, -1.6666654611e-1f), z * r, r);
  const float cp = fmaf(fmaf(fmaf(2.443315711809948e-5f, z, -1.388731625493765e-3f), z, 4.166664568298827e-2f), z * z,
                        fmaf(-0.5f, z, 1.0f));
  const int q = (int)k;
  const float s0 = (q & 1) ? cp : sp, c0 = (q & 1) ? sp : cp;
  *sn = (q & 2) ? -s0 : s0;
  *cn = ((q + 1) & 2) ? -c0 : c0;
}
__device__ __forceinline__ float rsqrt_fast(float x) {  // MUFU.RSQ; the operands here are normal numbers
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// atan2 for the bearing residual: octant reduction to |t| <= tan(pi/8) with ONE approximate division
// (t = min/max, or (min - max)/(min + max) shifted by pi/4) and the single-precision minimax kernel of
// Cephes atanf; ~2e-7 rad absolute, a third of the instructions of atan2f (57 per call with the wrap,
// measured: the largest single line of the assembly).  atan2(0, 0) = 0.
__device__ __forceinline__ float atan2_fast(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  const bool big = mn > 0.41421356237f * mx;
  const float num = big ? mn - mx : mn, den = fmaxf(big ? mn + mx : mx, 1e-30f);
  const float t = __fdividef(num, den);
  const float z = t * t;
  float r = fmaf(fmaf(fmaf(fmaf(8.05374449538e-2f, z, -1.38776856032e-1f), z, 1.99777106478e-1f), z, -3.33329491539e-1f) * z, t, t);
  if (big) r += 0.78539816339744831f;
  if (ay > ax) r = 1.5707963267948966f - r;
  if (x < 0.f) r = 3.1415926535897932f - r;
  return copysignf(r, y);
}
__device__ __forceinline__ uint64_t lowmask(int k) { return k >= 64 ? ~0ull : ((1ull << k) - 1ull); }
__device__ __forceinline__ uint64_t ring_to_slot(uint64_t ring, int head, int W) {
  const uint64_t mW = lowmask(W);
  ring &= mW;
  if (head == 0) return ring;
  return ((ring >> head) | (ring << (W - head))) & mW;
}
__device__ __forceinline__ uint64_t slot_to_ring(uint64_t slot, int head, int W) {
  const uint64_t mW = lowmask(W);
  slot &= mW;
  if (head == 0) return slot;
  return ((slot << head) | (slot >> (W - head))) & mW;
}
__device__ __forceinline__ int nth_set_bit(uint64_t m, int k) {  // k-th (0-based) set bit; tiny code on purpose
#pragma unroll 1
  for (int i = 0; i < k; ++i) m &= m - 1;
  return __ffsll((long long)m) - 1;
}
// index of the k-th (0-based) set bit of a 32-bit word, by bisection on popcounts (k < popc(m))
__device__ __forceinline__ int nth_bit32(uint32_t m, int k) {
  int r = 0;
#pragma unroll
  for (int h = 16; h > 0; h >>= 1) {
    const int t = __popc(m & ((1u << h) - 1u));
    if (k >= t) { k -= t; r += h; m >>= h; }
  }
  return r;
}
// (p, q) of the packed lower-triangular index t = p(p+1)/2 + q, q <= p
__device__ __forceinline__ int tri_row(int t) {
  int p = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
  if ((p + 1) * (p + 2) / 2 <= t) ++p;
  if (p * (p + 1) / 2 > t) --p;
  return p;
}
// (p, q) of packed index t -> of t + step, without the square root: q moves right and wraps over the row ends
__device__ __forceinline__ void tri_advance(int& p, int& q, int step) {
  q += step;
  while (q > p) { q -= p + 1; ++p; }
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
  return v;
}

// A TEAM of TEAM threads (1, 2 or 4 warps) owns one environment.  `lane` below is the thread index
// inside the team.  Synchronisation is __syncwarp for one warp, a named barrier otherwise.
template <int TEAM>
struct Team {
  int bar;     // named barrier id (1..15)
  float* scr;  // shared scratch, 64 floats: reductions, diagonal tile, counters of the symbolic phase
  static constexpr int NW = TEAM / 32;
  __device__ __forceinline__ void sync() const {
    if (TEAM == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(TEAM) : "memory");
  }
  // sum of N values over the team (every thread gets the result); uniform call sites only
  template <int N>
  __device__ __forceinline__ void sum_n(float (&v)[N], int lane) const {
#pragma unroll
    for (int t = 0; t < N; ++t) v[t] = warp_sum(v[t]);
    if (TEAM > 32) {
      sync();
      if ((lane & 31) == 0) {
#pragma unroll
        for (int t = 0; t < N; ++t) scr[(lane >> 5) * N + t] = v[t];
      }
      sync();
#pragma unroll
      for (int t = 0; t < N; ++t) {
        float a = 0.f;
#pragma unroll
        for (int q = 0; q < NW; ++q) a += scr[q * N + t];
        v[t] = a;
      }
    }
  }
  __device__ __forceinline__ int min_int(int v, int lane) const {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(FULLMASK, v, o));
    if (TEAM > 32) {
      int* is = reinterpret_cast<int*>(scr);
      sync();
      if ((lane & 31) == 0) is[lane >> 5] = v;
      sync();
#pragma unroll
      for (int q = 0; q < NW; ++q) v = min(v, is[q]);
    }
    return v;
  }
  __device__ __forceinline__ bool any(bool p, int lane) const {
    int v = __any_sync(FULLMASK, p) ? 1 : 0;
    if (TEAM > 32) {
      int* is = reinterpret_cast<int*>(scr);
      sync();
      if ((lane & 31) == 0) is[lane >> 5] = v;
      sync();
#pragma unroll
      for (int q = 0; q < NW; ++q) v |= is[q];
    }
    return v != 0;
  }
};

__device__ __forceinline__ int ring_of(int slot, int head, int W) { int r = head + slot; return r >= W ? r - W : r; }
// state array index
__device__ __forceinline__ int st_pose(int k) { return 3 + 3 * k; }
__device__ __forceinline__ int st_lm(const Layout& ly, int l) { return 3 + 3 * ly.W + 2 * l; }
// elimination offsets
// Per-environment elimination order: landmarks WITHOUT a live range-bearing factor in the window
// ("passive": coupled through the prior only, or never seen) come first, then the chain poses, then the
// observed landmarks, padding, the newest pose and the anchor.  obs = landmarks observed from any slot.
struct Ord { uint64_t obs; int npas; };
__device__ __forceinline__ int off_new(const Layout& ly) { return 3 * (ly.W - 2) + 2 * ly.L + ly.pad; }
__device__ __forceinline__ int off_a(const Layout& ly) { return 3 * (ly.W - 2) + 2 * ly.L + ly.pad + 3; }
__device__ __forceinline__ int off_lm(const Layout& ly, const Ord& od, int l) {
  const uint64_t below = lowmask(l);
  return ((od.obs >> l) & 1ull) ? 2 * od.npas + 3 * (ly.W - 2) + 2 * __popcll(od.obs & below)
                                : 2 * __popcll(~od.obs & below);
}
__device__ __forceinline__ int off_slot(const Layout& ly, const Ord& od, int k, int c) {
  return k == c - 1 ? off_new(ly) : 2 * od.npas + 3 * (k - 1);
}
__device__ __forceinline__ Ord make_ord(const Layout& ly, const uint32_t* rbm, int c) {
  uint64_t obs = 0ull;
  for (int k = 0; k < c; ++k) {
    obs |= (uint64_t)rbm[k * ly.nw];
    if (ly.nw > 1) obs |= (uint64_t)rbm[k * ly.nw + 1] << 32;
  }
  Ord od;
  od.obs = obs & lowmask(ly.L);
  od.npas = ly.L - __popcll(od.obs);
  return od;
}

struct Masks {  // warp-uniform
  uint64_t ps;   // prior support, pose SLOTS (bit k = slot k)
  uint64_t ls;   // prior support, landmarks
  uint64_t act;  // active landmarks
  uint64_t um;   // pose SLOTS with a unary absolute-pose factor
};

// ------------------------------------------------------------------ load / store of the record
template <int TEAM>
__device__ void load_env(const Layout& ly, const float* rec, const WS& w, const Team<TEAM>& tm, int lane, int head, int c, Masks& mk) {
  const int W = ly.W, L = ly.L;
  const int* reci = (const int*)rec;
  const uint32_t* recu = (const uint32_t*)rec;
  if (lane < 3) w.st[lane] = rec[ly.o_a + lane];
  for (int i = lane; i < 3 * W; i += TEAM) {
    const int k = i / 3, j = i - 3 * k, r = ring_of(k, head, W);
    const bool live = k < c;
    w.st[3 + i] = (live && k > 0) ? rec[ly.o_e + 3 * r + j] : 0.0f;
  }
  for (int k = lane; k < W; k += TEAM) {
    const int r = ring_of(k, head, W);
    const int t = (k < c) ? reci[ly.o_lct + r] : -1;
    int ts = -1;
    if (t >= 0) { ts = t - head; if (ts < 0) ts += W; }
    w.lct[k] = ts;
    for (int q = 0; q < ly.nw; ++q) w.rbm[k * ly.nw + q] = (k < c) ? recu[ly.o_rbm + r * ly.nw + q] : 0u;
  }
  for (int i = lane; i < 2 * L; i += TEAM) w.st[3 + 3 * W + i] = rec[ly.o_m + i];
  const uint64_t pm = (uint64_t)recu[ly.o_pm] | ((uint64_t)recu[ly.o_pm + 1] << 32);
  mk.ps = ring_to_slot(pm, head, W);
  mk.ls = (uint64_t)recu[ly.o_lm] | ((uint64_t)recu[ly.o_lm + 1] << 32);
  mk.act = (uint64_t)recu[ly.o_act] | ((uint64_t)recu[ly.o_act + 1] << 32);
  mk.um = ring_to_slot((uint64_t)recu[ly.o_um] | ((uint64_t)recu[ly.o_um + 1] << 32), head, W) & lowmask(c);
  {  // the prior (Lambda, g, vbar) is first needed by assemble, thousands of cycles from here: pull it into L2 now
    const int sp = 3 + 3 * __popcll(pm) + 2 * __popcll(mk.ls);
    const int nl = ((sp * (sp + 1) >> 1) + 31) >> 5;  // 128-byte lines of the packed triangle
    for (int i = lane; i < nl; i += TEAM) asm volatile("prefetch.global.L2 [%0];" ::"l"(rec + ly.o_lam + 32 * i));
    if (lane < ((sp + 31) >> 5)) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(rec + ly.o_g + 32 * lane));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(rec + ly.o_vbar + 32 * lane));
    }
  }
  tm.sync();
}

// writes a, e (ring positions of the CURRENT head), m, active mask
template <int TEAM>
__device__ void store_state(const Layout& ly, float* rec, const WS& w, const Team<TEAM>& tm, int lane, int head, int c, const Masks& mk) {
  const int W = ly.W, L = ly.L;
  uint32_t* recu = (uint32_t*)rec;
  if (lane < 3) rec[ly.o_a + lane] = w.st[lane];
  for (int i = lane; i < 3 * c; i += TEAM) {
    const int k = i / 3, j = i - 3 * k, r = ring_of(k, head, W);
    rec[ly.o_e + 3 * r + j] = w.st[3 + i];
  }
  for (int i = lane; i < 2 * L; i += TEAM) rec[ly.o_m + i] = w.st[3 + 3 * W + i];
  if (lane == 0) {
    recu[ly.o_act] = (uint32_t)mk.act; recu[ly.o_act + 1] = (uint32_t)(mk.act >> 32);
    const uint64_t um = slot_to_ring(mk.um, head, W);
    recu[ly.o_um] = (uint32_t)um; recu[ly.o_um + 1] = (uint32_t)(um >> 32);
  }
}

// ------------------------------------------------------------------ S0 push / observe
// Range-bearing bookkeeping for the pose in `slot` (pose px,py,pth in the anchor frame; landmarks are
// kept in GLOBAL coordinates, reading R17b).
template <int TEAM>
__device__ void record_rb(const Layout& ly, float* rec, const WS& w, const Team<TEAM>& tm, int lane, int env, int head, int slot,
                          float px, float py, float pth, const StepIO& io, Masks& mk) {
  const int L = ly.L, N = ly.N, r = ring_of(slot, head, ly.W);
  uint32_t* recu = (uint32_t*)rec;
  uint64_t vis = (uint64_t)io.rb_mask[env];
  if (ly.nw > 1) vis |= (uint64_t)io.rb_mask[(size_t)N + env] << 32;
  vis &= lowmask(L);
  for (int l = lane; l < L; l += TEAM) {
    const float zr = io.rb_meas[(size_t)l * N + env];
    const float zb = io.rb_meas[(size_t)(L + l) * N + env];
    rec[ly.o_zrb + (r * 2 + 0) * L + l] = zr;
    rec[ly.o_zrb + (r * 2 + 1) * L + l] = zb;
    if (((vis >> l) & 1ull) && !((mk.act >> l) & 1ull)) {  // R6: inverse projection from the observing pose's guess (global)
      float sa, ca, sn, cn;
      sincos_pi(w.st[2], &sa, &ca);
      const float gx = w.st[0] + ca * px - sa * py, gy = w.st[1] + sa * px + ca * py;
      sincos_pi(w.st[2] + pth + zb, &sn, &cn);
      w.st[st_lm(ly, l)] = gx + zr * cn;
      w.st[st_lm(ly, l) + 1] = gy + zr * sn;
    }
  }
  if (lane < ly.nw) {
    const uint32_t word = (uint32_t)(vis >> (32 * lane));
    w.rbm[slot * ly.nw + lane] = word;
    recu[ly.o_rbm + r * ly.nw + lane] = word;
  }
  mk.act |= vis;
  tm.sync();
}

// Appends slot c (count before the push).  Returns the new count.
template <int TEAM>
__device__ int push_env(const Layout& ly, float* rec, const WS& w, const Team<TEAM>& tm, int lane, int env, int head, int c,
                        const StepIO& io, Masks& mk) {
  const int W = ly.W, N = ly.N, r = ring_of(c, head, W);
  int* reci = (int*)rec;
  const float zx = io.odom[env], zy = io.odom[(size_t)N + env], zt = io.odom[2 * (size_t)N + env];
  const float* p = w.st + st_pose(c - 1);  // slot 0 is stored as zeros
  const float pxo = p[0], pyo = p[1], pto = p[2];
  float sn, cn;
  sincos_pi(pto, &sn, &cn);
  const float nx = pxo + cn * zx - sn * zy, ny = pyo + sn * zx + cn * zy, nt = wrapf(pto + zt);
  int back = io.lc_back ? io.lc_back[env] : 0;
  const int tgt = (back >= 1 && back <= c) ? c - back : -1;  // R11
  tm.sync();
  if (lane == 0) {
    float* q = w.st + st_pose(c);
    q[0] = nx; q[1] = ny; q[2] = nt;
    w.lct[c] = tgt;
    reci[ly.o_lct + r] = tgt < 0 ? -1 : ring_of(tgt, head, W);
  }
  if (lane < 3) {
    const float z = lane == 0 ? zx : (lane == 1 ? zy : zt);
    rec[ly.o_zodo + 3 * r + lane] = z;   // (measurements stay in the record: read from L2 once per linearisation)
    const float zl = io.lc_meas ? io.lc_meas[(size_t)lane * N + env] : 0.0f;
    rec[ly.o_zlc + 3 * r + lane] = zl;
  }
  mk.um &= ~(1ull << c);
  if (io.un_pose && (io.un_valid == nullptr || io.un_valid[env] != 0)) {
    if (lane < 3) rec[ly.o_zun + 3 * r + lane] = io.un_pose[(size_t)lane * N + env];
    if (lane < 6) rec[ly.o_omun + 6 * r + lane] = io.un_info[(size_t)lane * N + env];
    mk.um |= 1ull << c;
  }
  tm.sync();
  if (ly.L > 0) record_rb<TEAM>(ly, rec, w, tm, lane, env, head, c, nx, ny, nt, io, mk);
  return c + 1;
}

// ------------------------------------------------------------------ prior support tables
// For support scalar p (canonical order [a | poses by slot | landmarks]): elimination offset in
// ssup[p], state index in sidx[p] (bit 16 set for angle components).  Returns the support dimension.
template <int TEAM>
__device__ int build_support(const Layout& ly, const Ord& od, const WS& w, const Team<TEAM>& tm, int lane, int c, uint64_t ps, uint64_t ls) {
  const int npo = __popcll(ps), nlo = __popcll(ls);
  const int s = 3 + 3 * npo + 2 * nlo;
  for (int p = lane; p < s; p += TEAM) {
    int off, idx;
    if (p < 3) { off = off_a(ly) + p; idx = p | (p == 2 ? 0x10000 : 0); }
    else if (p < 3 + 3 * npo) {
      const int b = (p - 3) / 3, j = (p - 3) - 3 * b, k = nth_set_bit(ps, b);
      off = off_slot(ly, od, k, c) + j; idx = (st_pose(k) + j) | (j == 2 ? 0x10000 : 0);
    } else {
      const int q = p - 3 - 3 * npo, b = q >> 1, j = q & 1, l = nth_set_bit(ls, b);
      off = off_lm(ly, od, l) + j; idx = st_lm(ly, l) + j;
    }
    w.sup[p] = (uint32_t)off | ((uint32_t)(idx & 0xffff) << 9) | ((idx & 0x10000) ? (1u << 18) : 0u);
  }
  tm.sync();
  return s;
}

// ------------------------------------------------------------------ symbolic phase: envelope of H
// Rows are grouped in pairs; both rows of a pair store the columns [first, 4g+3] of their tile row g (whole 4x4 tiles,
// first a multiple of 4), so every tile row is one aligned 128-bit word.  first[i] = first column
// of row i; rbase[i] + j addresses H(i,j).  Row np (the rhs; index np+1 is an alias of it) spans [0, np).
// Returns the total words used.
template <int TEAM>
__device__ int symbolic(const Layout& ly, const Ord& od, const WS& w, const Team<TEAM>& tm, int lane, int c, const Masks& mk, int s) {
  const int L = ly.L, np = ly.np;
  const int oC = 2 * od.npas, oL = oC + 3 * (ly.W - 2), oP = 3 * (ly.W - 2) + 2 * L, oN = off_new(ly), oA = off_a(ly);
  int* tfirst = reinterpret_cast<int*>(w.sds);  // first column per row while it is being built (sds is free until assemble)
  // own block offsets
  for (int i = lane; i < np + 2; i += TEAM) {
    int f;
    if (i < oC) f = i & ~1;
    else if (i < oL) f = oC + ((i - oC) / 3) * 3;
    else if (i < oP) f = oL + ((i - oL) >> 1) * 2;
    else if (i < oN) f = i;
    else if (i < oA) f = oN;
    else if (i < np) f = oA;
    else f = 0;
    tfirst[i] = f;
  }
  tm.sync();
  // pose rows
  for (int k = 1 + lane; k < c; k += TEAM) {
    const int o = off_slot(ly, od, k, c);
    int f = o;
    if (k >= 2) f = min(f, off_slot(ly, od, k - 1, c));
    const int t = w.lct[k];
    if (t >= 1) f = min(f, off_slot(ly, od, t, c));
    if (k == c - 1 && L > 0) {  // newest pose comes after the landmarks it observes
      uint64_t m = (uint64_t)w.rbm[k * ly.nw];
      if (ly.nw > 1) m |= (uint64_t)w.rbm[k * ly.nw + 1] << 32;
      if (m) f = min(f, off_lm(ly, od, __ffsll((long long)m) - 1));
    }
    tfirst[o] = f; tfirst[o + 1] = f; tfirst[o + 2] = f;
  }
  // landmark rows: first chain pose (slots 1..c-2) that observes them
  for (int l = lane; l < L; l += TEAM) {
    const int o = off_lm(ly, od, l);
    int f = o;
    for (int k = 1; k <= c - 2; ++k)
      if ((w.rbm[k * ly.nw + (l >> 5)] >> (l & 31)) & 1u) { f = oC + 3 * (k - 1); break; }
    tfirst[o] = f; tfirst[o + 1] = f;
  }
  tm.sync();
  // prior: all support blocks are mutually coupled
  if (s > 3) {
    int fs = np;
    for (int p = 3 + lane; p < s; p += TEAM) fs = min(fs, sup_off(w.sup[p]));
    fs = tm.min_int(fs, lane);
    for (int p = lane; p < s; p += TEAM) { const int i = sup_off(w.sup[p]); tfirst[i] = min(tfirst[i], fs); }
  }
  tm.sync();
  // landmarks are global: every range-bearing factor also touches the anchor, whose rows therefore
  // reach back to the first observing chain pose and the first observed landmark
  if (L > 0) {
    int fa = oA;
    for (int k = lane; k < c; k += TEAM) {
      uint64_t m = (uint64_t)w.rbm[k * ly.nw];
      if (ly.nw > 1) m |= (uint64_t)w.rbm[k * ly.nw + 1] << 32;
      if (m) {
        if (k >= 1) fa = min(fa, off_slot(ly, od, k, c));
        fa = min(fa, off_lm(ly, od, __ffsll((long long)m) - 1));
      }
    }
    fa = tm.min_int(fa, lane);
    if (lane < 3) tfirst[oA + lane] = min(tfirst[oA + lane], fa);
  }
  tm.sync();
  if (mk.um >> 1) {  // unary factors couple the anchor to their pose (x_k = a (+) e_k)
    const int kmin = __ffsll((long long)(mk.um >> 1));  // lowest slot >= 1
    if (lane < 3) tfirst[oA + lane] = min(tfirst[oA + lane], off_slot(ly, od, kmin, c));
    tm.sync();
  }
  // group rows in fours, or (ly.pairs) in PAIRS (shared first, aligned down to 4: whole 4x4 tile rows);
  // prefix sum of the row lengths -> rbase (done by the first warp of the team).  A pair is what one
  // lane of the factorisation owns; with pairs the two pairs of a 4-column block may start at different
  // columns (cholesky<.., true> splits its dot products there), which stores 12-18 % fewer words than a
  // common start for all four rows at ~30 more instructions per column block: worth it where shared
  // memory bounds the environments in flight (slam_api.cu: pick_pairs).
  if (lane < 32) {
    int run = 0;
    for (int base = 0; base < np + 2; base += 32) {
      const int i = base + lane;
      int f = 0, len = 0;
      if (i < np) {
        if (ly.pairs) {
          const int g2 = i & ~1;
          f = min(tfirst[g2], tfirst[g2 + 1]) & ~3;
        } else {
          const int g4 = i & ~3;
          f = min(min(tfirst[g4], tfirst[g4 + 1]), min(tfirst[g4 + 2], tfirst[g4 + 3])) & ~3;
        }
        len = (i | 3) + 1 - f;
      } else if (i == np) {   // the rhs row; its pair twin (row np + 1) is the SAME storage, see build_lists
        len = np;
      }
      int x = len;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULLMASK, x, o); if (lane >= o) x += y; }
      __syncwarp();
      if (i < np + 2) w.rbf[i] = (uint32_t)(run + x - (i == np + 1 ? np : len) - f) | ((uint32_t)(f >> 2) << 16);
      run += __shfl_sync(FULLMASK, x, 31);
    }
    if (lane == 0) reinterpret_cast<int*>(tm.scr)[8] = run;
  }
  tm.sync();
  if (lane < 32) {  // loop-closure mask for assemble
    const uint32_t lo = __ballot_sync(FULLMASK, lane < c && w.lct[lane] >= 0);
    const uint32_t hi = __ballot_sync(FULLMASK, lane + 32 < c && w.lct[lane + 32] >= 0);
    if (lane == 0) { w.lct[ly.W] = (int)lo; w.lct[ly.W + 1] = (int)hi; }
  }
  // words of the active-pair lists (build_lists): pair p (rows 2p, 2p+1; the rhs pair is p = np/2) is
  // active in the column blocks J with first <= 4J <= 2p, so the list sizes follow from first[] alone
  if (lane < 32) {
    const int G = np >> 2, NP = (np >> 1) + 1;
    int cntp = 0;
    for (int p = lane; p < NP; p += 32) cntp += min(p >> 1, G - 1) - (first_of(w, 2 * p) >> 2) + 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cntp += __shfl_xor_sync(FULLMASK, cntp, o);
    if (lane == 0) reinterpret_cast<int*>(tm.scr)[10] = (G + 1) + NP + ((cntp + 3) >> 2) + 3 & ~3;
  }
  tm.sync();
  return reinterpret_cast<const int*>(tm.scr)[8];
}

// Second part of the symbolic phase, after the environment got its share of the pool (w.amask is set):
// the tables the factorisation walks, so that one shared-memory load per column block and one per lane
// replace the chains of dependent index look-ups (measured: ~280 instructions of fixed cost per block).
//   hdr[J]   (G+1 words)  offset of the block's list (14 bit) | pairs in it (8 bit) | K-split log2 for
//                         teams of 32 / 64 / 128 threads (2 bit each)
//   ptab[p]  (NP words)   row pair p (rows 2p, 2p+1 of one 4-row group; p = np/2 is the rhs pair):
//                         start of row 2p in H / 4 (14 bit) | first / 4 (7 bit) | row length / 4 (7 bit)
//   alist    (bytes)      active pairs per 4-column block J: pair p takes part in column J iff
//                         first <= 4J <= 2p; ascending, so the two diagonal pairs 2J, 2J+1 come first
// Built by the first warp.
struct Tables { const uint32_t* hdr; const uint32_t* ptab; const unsigned char* alist; };
__device__ __forceinline__ Tables tables_of(const Layout& ly, const WS& w) {
  Tables t;
  t.hdr = w.amask;
  t.ptab = w.amask + (ly.np >> 2) + 1;
  t.alist = reinterpret_cast<const unsigned char*>(t.ptab + (ly.np >> 1) + 1);
  return t;
}
template <int TEAM>
__device__ void build_lists(const Layout& ly, const WS& w, const Team<TEAM>& tm, int lane) {
  const int np = ly.np;
  if (lane < 32) {
    const int G = np >> 2, NP = (np >> 1) + 1;
    uint32_t* hdr = w.amask;
    uint32_t* ptab = hdr + G + 1;
    unsigned char* alist = reinterpret_cast<unsigned char*>(ptab + NP);
    for (int p = lane; p < NP; p += 32) {
      // the rhs "pair" is the rhs row twice (length 0 between its rows): both lanes' results are the same
      // bits written to the same words, and no zero twin row has to be stored
      const int i = 2 * p, f = first_of(w, i), len = i < np ? (i | 3) + 1 - f : 0;
      ptab[p] = (uint32_t)((rb_of(w, i) + f) >> 2) | ((uint32_t)(f >> 2) << 14) | ((uint32_t)(len >> 2) << 21);
    }
    int run = 0, maxcnt = 0;
    for (int J = 0; J < G; ++J) {
      const int start = run;
      for (int base = 2 * J; base < NP; base += 32) {
        const int p = base + lane;
        const bool on = p < NP && first_of(w, 2 * p) <= 4 * J;
        const uint32_t bal = __ballot_sync(FULLMASK, on);
        if (on) alist[run + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)p;
        run += __popc(bal);
      }
      const int cnt = run - start;
      maxcnt = max(maxcnt, cnt);
      if (lane == 0) {
        // K-split: when a column has fewer pairs than threads, 2^lg adjacent lanes share one pair and split
        // its dot-product range; only worth it when the dot products are long
        uint32_t lgs = 0;
        if (4 * J - min(first_of(w, 4 * J), first_of(w, 4 * J + 2)) >= SLAM_KSPLIT_MIN) {
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            if (q != 0 && (32 << q) != TEAM) continue;   // only the team sizes this kernel factorises with
            int lg = 0;
            while (lg < 3 && (cnt << (lg + 1)) <= (32 << q)) ++lg;
            lgs |= (uint32_t)lg << (2 * q);
          }
        }
        hdr[J] = (uint32_t)start | ((uint32_t)cnt << 14) | (lgs << 22);
      }
    }
    if (lane == 0) { hdr[G] = (uint32_t)run; reinterpret_cast<int*>(tm.scr)[9] = maxcnt; }
  }
  tm.sync();
}

// ------------------------------------------------------------------ S1 + S2: linearise and assemble
struct Between {  // residual and the pieces of J_i, J_j of a between factor (A.2)
  float r[3], c, s, hx, hy;
};
__device__ __forceinline__ Between between_eval(const float* pi, float ci, float si, const float* pj, const float* z) {
  Between b;
  const float dx = pj[0] - pi[0], dy = pj[1] - pi[1];
  b.c = ci; b.s = si;
  b.hx = ci * dx + si * dy; b.hy = -si * dx + ci * dy;
  b.r[0] = b.hx - z[0]; b.r[1] = b.hy - z[1]; b.r[2] = wrapf(pj[2] - pi[2] - z[2]);
  return b;
}
// J_j = [[c,s,0],[-s,c,0],[0,0,1]],  J_i = [[-c,-s,hy],[s,-c,-hx],[0,0,-1]]
__device__ __forceinline__ void between_jac(const Between& b, float Ji[3][3], float Jj[3][3]) {
  Jj[0][0] = b.c; Jj[0][1] = b.s; Jj[0][2] = 0.f;
  Jj[1][0] = -b.s; Jj[1][1] = b.c; Jj[1][2] = 0.f;
  Jj[2][0] = 0.f; Jj[2][1] = 0.f; Jj[2][2] = 1.f;
  Ji[0][0] = -b.c; Ji[0][1] = -b.s; Ji[0][2] = b.hy;
  Ji[1][0] = b.s; Ji[1][1] = -b.c; Ji[1][2] = -b.hx;
  Ji[2][0] = 0.f; Ji[2][1] = 0.f; Ji[2][2] = -1.f;
}

// H(rowblock oj, colblock oi) += Jj' Om Ji (full 3x3), H(oj,oj) += Jj' Om Jj (lower), b(oj) -= Jj' Om r
__device__ __forceinline__ void add_j_side(const WS& w, int n, int oj, int oi, const float Ji[3][3], const float Jj[3][3],
                                           const float* om, const float* r, bool has_i) {
  float* rhs = w.H + rb_of(w, n);
#pragma unroll
  for (int x = 0; x < 3; ++x) {
    float* row = w.H + rb_of(w, oj + x);
    float g = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) g = fmaf(Jj[k][x] * om[k], r[k], g);
    rhs[oj + x] -= g;
#pragma unroll
    for (int y = 0; y <= x; ++y) {
      float h = 0.f;
#pragma unroll
      for (int k = 0; k < 3; ++k) h = fmaf(Jj[k][x] * om[k], Jj[k][y], h);
      row[oj + y] += h;
    }
    if (has_i) {
#pragma unroll
      for (int y = 0; y < 3; ++y) {
        float h = 0.f;
#pragma unroll
        for (int k = 0; k < 3; ++k) h = fmaf(Jj[k][x] * om[k], Ji[k][y], h);
        row[oi + y] += h;
      }
    }
  }
}
__device__ __forceinline__ void acc_i_side(const float Ji[3][3], const float* om, const float* r, float Hii[6], float gi[3]) {
  int t = 0;
#pragma unroll
  for (int x = 0; x < 3; ++x) {
#pragma unroll
    for (int k = 0; k < 3; ++k) gi[x] = fmaf(Ji[k][x] * om[k], r[k], gi[x]);
#pragma unroll
    for (int y = 0; y <= x; ++y) {
#pragma unroll
      for (int k = 0; k < 3; ++k) Hii[t] = fmaf(Ji[k][x] * om[k], Ji[k][y], Hii[t]);
      ++t;
    }
  }
}
__device__ __forceinline__ void add_i_side(const WS& w, int n, int oi, const float Hii[6], const float gi[3]) {
  float* rhs = w.H + rb_of(w, n);
  int t = 0;
#pragma unroll
  for (int x = 0; x < 3; ++x) {
    float* row = w.H + rb_of(w, oi + x);
    rhs[oi + x] -= gi[x];
#pragma unroll
    for (int y = 0; y <= x; ++y) row[oi + y] += Hii[t++];
  }
}

// Builds H and b (row n) at the current state.  `s` = prior support dimension.
template <int TEAM>
__device__ void assemble(const Layout& ly, const Params& pr, const Ord& od, const float* rec, const WS& w, const Team<TEAM>& tm, int lane, int head,
                         int c, const Masks& mk, int s, int total, int cb) {
  const int W = ly.W, L = ly.L, n = ly.np;  // n: row index of the rhs
  // cb > 0 (second and later linearisation of one call): the columns [0, cb) -- passive landmarks, which
  // only the constant prior touches -- still hold their factor L from the previous factorisation; they are
  // kept (see cholesky) and only the columns >= cb and the rhs rows are rebuilt.
  if (cb == 0) {
    for (int t = lane; t < total; t += TEAM) w.H[t] = 0.f;
  } else {
    for (int i = lane; i < n + 2; i += TEAM) {
      const int lo = i < n ? max(first_of(w, i), cb) : 0, hi = i < n ? (i | 3) + 1 : n;  // (the rhs rows span [0, n))
      float4* z = reinterpret_cast<float4*>(w.H + rb_of(w, i) + lo);
      for (int t = 0; t < (hi - lo) >> 2; ++t) z[t] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  // cos/sin of every live pose (slot 0 is the frame itself)
  for (int k = lane; k < c; k += TEAM) {
    float sn = 0.f, cn = 1.f;
    if (k > 0) sincos_pi(w.st[st_pose(k) + 2], &sn, &cn);
    w.cs[2 * k] = cn; w.cs[2 * k + 1] = sn;
  }
  // prior displacement d = v - vbar on the support (angles wrapped)
  bool dnz = false;  // any non-zero displacement?  (none at the first linearisation after a marginalisation)
  for (int p = lane; p < s; p += TEAM) {
    const uint32_t e = w.sup[p];
    float d = w.st[sup_idx(e)] - rec[ly.o_vbar + p];
    if (sup_angle(e)) d = wrapf(d);
    w.sds[p] = d;
    dnz |= d != 0.0f;
  }
  dnz = tm.any(dnz, lane);
  tm.sync();
  // identity rows for unused chain slots, the unused newest slot (c == 1), inactive landmarks, padding
  for (int k = max(c - 1, 1) + lane; k <= W - 2; k += TEAM) {
    const int o = 2 * od.npas + 3 * (k - 1);
    w.H[rb_of(w, o) + o] = 1.0f; w.H[rb_of(w, o + 1) + o + 1] = 1.0f; w.H[rb_of(w, o + 2) + o + 2] = 1.0f;
  }
  for (int l = lane; l < L; l += TEAM)
    if (!((mk.act >> l) & 1ull)) {
      const int o = off_lm(ly, od, l);
      if (o >= cb) { w.H[rb_of(w, o) + o] = 1.0f; w.H[rb_of(w, o + 1) + o + 1] = 1.0f; }
    }
  if (lane < ly.pad + (c < 2 ? 3 : 0)) {
    const int o = off_new(ly) - ly.pad + lane;
    w.H[rb_of(w, o) + o] = 1.0f;
  }
  // prior: H += Lambda (row by row, coalesced over the packed lower triangle)
  {
    const float* lam = rec + ly.o_lam;
    // flat over the packed triangle: coalesced, and every iteration is independent (memory-level
    // parallelism: the loads of Lambda come from L2)
    const int ntri = s * (s + 1) >> 1;
    // loads first, scatter second: the compiler cannot move a global load above the shared-memory update
    // of the previous entry, so without the explicit batch every iteration pays a full L2 round trip
    int tp = tri_row(lane), tq = lane - (tp * (tp + 1) >> 1);   // (row, column) of this lane's entry, advanced incrementally
    for (int t0 = lane; t0 < ntri; t0 += 8 * TEAM) {
      float v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) { const int t = t0 + u * TEAM; v[u] = t < ntri ? lam[t] : 0.f; }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int t = t0 + u * TEAM;
        if (t < ntri) {
          const int ip = sup_off(w.sup[tp]), iq = sup_off(w.sup[tq]);
          const int hi = max(ip, iq), lo = min(ip, iq);
          if (lo >= cb) w.H[rb_of(w, hi) + lo] += v[u];
          tri_advance(tp, tq, TEAM);
        }
      }
    }
    // b -= Lambda d + g (row p: the packed row, then the column below the diagonal; 8 loads in flight)
    float* rhs = w.H + rb_of(w, n);
    for (int p = lane; p < s; p += TEAM) {
      float acc0 = rec[ly.o_g + p], acc1 = 0.f;
      const float* lrow = lam + (p * (p + 1) >> 1);
      if (!dnz) { rhs[sup_off(w.sup[p])] -= acc0; continue; }  // Lambda d = 0: the same value without the products
      for (int q0 = 0; q0 <= p; q0 += 8) {
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = q0 + u <= p ? lrow[q0 + u] : 0.f;
#pragma unroll
        for (int u = 0; u < 8; u += 2) {
          acc0 = fmaf(v[u], q0 + u <= p ? w.sds[q0 + u] : 0.f, acc0);
          acc1 = fmaf(v[u + 1], q0 + u + 1 <= p ? w.sds[q0 + u + 1] : 0.f, acc1);
        }
      }
      for (int q0 = p + 1; q0 < s; q0 += 8) {
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) { const int q = q0 + u; v[u] = q < s ? lam[(q * (q + 1) >> 1) + p] : 0.f; }
#pragma unroll
        for (int u = 0; u < 8; u += 2) {
          acc0 = fmaf(v[u], q0 + u < s ? w.sds[q0 + u] : 0.f, acc0);
          acc1 = fmaf(v[u + 1], q0 + u + 1 < s ? w.sds[q0 + u + 1] : 0.f, acc1);
        }
      }
      rhs[sup_off(w.sup[p])] -= acc0 + acc1;
    }
  }
  tm.sync();
  // odometry factors k-1 -> k: phase A (j side), phase B (i side)
  for (int pass = 0; pass < 2; ++pass) {
    for (int k = 1 + lane; k < c; k += TEAM) {
      const float* pi = w.st + st_pose(k - 1);
      const float* pj = w.st + st_pose(k);
      const Between b = between_eval(pi, w.cs[2 * (k - 1)], w.cs[2 * (k - 1) + 1], pj, rec + ly.o_zodo + 3 * ring_of(k, head, W));
      float Ji[3][3], Jj[3][3];
      between_jac(b, Ji, Jj);
      if (pass == 0) {
        add_j_side(w, n, off_slot(ly, od, k, c), k >= 2 ? off_slot(ly, od, k - 1, c) : 0, Ji, Jj, pr.om_odo, b.r, k >= 2);
      } else if (k >= 2) {
        float Hii[6] = {0, 0, 0, 0, 0, 0}, gi[3] = {0, 0, 0};
        acc_i_side(Ji, pr.om_odo, b.r, Hii, gi);
        add_i_side(w, n, off_slot(ly, od, k - 1, c), Hii, gi);
      }
    }
    tm.sync();
  }
  // loop closures t -> k: phase C (j side: at most one per k), phase D (i side: lane per target).
  // lcm (bit k: slot k closes a loop; from the symbolic phase) skips both when there is none and
  // bounds the search of phase D.
  const uint64_t lcm = (uint64_t)(uint32_t)w.lct[W] | ((uint64_t)(uint32_t)w.lct[W + 1] << 32);
  if (lcm) {
    for (int k = 1 + lane; k < c; k += TEAM) {
      const int t = w.lct[k];
      if (t < 0) continue;
      const Between b = between_eval(w.st + st_pose(t), w.cs[2 * t], w.cs[2 * t + 1], w.st + st_pose(k), rec + ly.o_zlc + 3 * ring_of(k, head, W));
      float Ji[3][3], Jj[3][3];
      between_jac(b, Ji, Jj);
      add_j_side(w, n, off_slot(ly, od, k, c), t >= 1 ? off_slot(ly, od, t, c) : 0, Ji, Jj, pr.om_lc, b.r, t >= 1);
    }
    tm.sync();
    for (int t = 1 + lane; t < c - 1; t += TEAM) {
      float Hii[6] = {0, 0, 0, 0, 0, 0}, gi[3] = {0, 0, 0};
      bool any = false;
      uint64_t km = lcm & ~((2ull << t) - 1ull);
      while (km) {
        const int k = __ffsll((long long)km) - 1;
        km &= km - 1;
        if (w.lct[k] != t) continue;
        const Between b = between_eval(w.st + st_pose(t), w.cs[2 * t], w.cs[2 * t + 1], w.st + st_pose(k), rec + ly.o_zlc + 3 * ring_of(k, head, W));
        float Ji[3][3], Jj[3][3];
        between_jac(b, Ji, Jj);
        acc_i_side(Ji, pr.om_lc, b.r, Hii, gi);
        any = true;
      }
      if (any) add_i_side(w, n, off_slot(ly, od, t, c), Hii, gi);
    }
    tm.sync();
  }
  // unary absolute-pose factors (NEXT-1): r = (a (+) e_k) - z, full 3x3 information,
  // J_a = [[1,0,-dy],[0,1,dx],[0,0,1]] (d = Rot(a_th) t_k), J_e = blockdiag(Rot(a_th), 1); slot 0: x = a.
  if (mk.um) {
    float* rhs = w.H + rb_of(w, n);
    const int oA = off_a(ly);
    float sa, ca;
    sincos_pi(w.st[2], &sa, &ca);
    float A[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};  // anchor block (lower 6) and gradient (3)
    for (int k = lane; k < c; k += TEAM) {
      if (!((mk.um >> k) & 1ull)) continue;
      const int r = ring_of(k, head, W);
      const float* e = w.st + st_pose(k);
      const float dx = ca * e[0] - sa * e[1], dy = sa * e[0] + ca * e[1];
      const float r0 = w.st[0] + dx - rec[ly.o_zun + 3 * r], r1 = w.st[1] + dy - rec[ly.o_zun + 3 * r + 1];
      const float r2 = wrapf(w.st[2] + e[2] - rec[ly.o_zun + 3 * r + 2]);
      const float* om = rec + ly.o_omun + 6 * r;
      const float O[3][3] = {{om[0], om[1], om[3]}, {om[1], om[2], om[4]}, {om[3], om[4], om[5]}};
      const float Ja[3][3] = {{1.f, 0.f, -dy}, {0.f, 1.f, dx}, {0.f, 0.f, 1.f}};
      const float Je[3][3] = {{ca, -sa, 0.f}, {sa, ca, 0.f}, {0.f, 0.f, 1.f}};
      float Or[3], OJa[3][3], OJe[3][3];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        Or[i] = O[i][0] * r0 + O[i][1] * r1 + O[i][2] * r2;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          OJa[i][j] = O[i][0] * Ja[0][j] + O[i][1] * Ja[1][j] + O[i][2] * Ja[2][j];
          OJe[i][j] = O[i][0] * Je[0][j] + O[i][1] * Je[1][j] + O[i][2] * Je[2][j];
        }
      }
      int t = 0;
#pragma unroll
      for (int x = 0; x < 3; ++x) {
#pragma unroll
        for (int y = 0; y <= x; ++y) A[t++] += Ja[0][x] * OJa[0][y] + Ja[1][x] * OJa[1][y] + Ja[2][x] * OJa[2][y];
        A[6 + x] += Ja[0][x] * Or[0] + Ja[1][x] * Or[1] + Ja[2][x] * Or[2];
      }
      if (k >= 1) {
        const int op = off_slot(ly, od, k, c);
#pragma unroll
        for (int x = 0; x < 3; ++x) {
          float* row = w.H + rb_of(w, op + x);
          float* arow = w.H + rb_of(w, oA + x);
#pragma unroll
          for (int y = 0; y <= x; ++y) row[op + y] += Je[0][x] * OJe[0][y] + Je[1][x] * OJe[1][y] + Je[2][x] * OJe[2][y];
#pragma unroll
          for (int y = 0; y < 3; ++y) arow[op + y] += Ja[0][x] * OJe[0][y] + Ja[1][x] * OJe[1][y] + Ja[2][x] * OJe[2][y];
          rhs[op + x] -= Je[0][x] * Or[0] + Je[1][x] * Or[1] + Je[2][x] * Or[2];
        }
      }
    }
    tm.sync();
    tm.sum_n(A, lane);
    if (lane == 0) {
      float* qa0 = w.H + rb_of(w, oA);
      float* qa1 = w.H + rb_of(w, oA + 1);
      float* qa2 = w.H + rb_of(w, oA + 2);
      qa0[oA] += A[0]; qa1[oA] += A[1]; qa1[oA + 1] += A[2];
      qa2[oA] += A[3]; qa2[oA + 1] += A[4]; qa2[oA + 2] += A[5];
      rhs[oA] -= A[6]; rhs[oA + 1] -= A[7]; rhs[oA + 2] -= A[8];
    }
    tm.sync();
  }
  // range-bearing factors.  Landmarks g are global, so each factor has three blocks: anchor a, observing
  // pose e_k (k >= 1), landmark g.  With the anchor-frame landmark m = Rot(a_th)'(g - a_t), D = m - t_k:
  //   J_e = [-J_l | (0,-1)'],  J_g = J_l Rot(a_th)',  J_a = [-J_g | -J_l S m].
  // Two passes, no cross-lane reductions inside the loops: pass A has one lane per POSE (sums over its
  // landmarks stay in registers: pose diagonal, gradient, anchor x pose block); pass B one lane per
  // LANDMARK (landmark diagonal, gradient, anchor x landmark block, anchor diagonal partial sums).
  if (L > 0 && od.obs) {
    float* rhs = w.H + rb_of(w, n);
    const float w0 = pr.om_rb[0], w1 = pr.om_rb[1];
    const int oA = off_a(ly);
    float sa, ca;
    sincos_pi(w.st[2], &sa, &ca);
    const float ax = w.st[0], ay = w.st[1];
    float* mloc = w.sds + s;  // anchor-frame landmark positions (2L floats after the prior displacement)
    for (int l = lane; l < L; l += TEAM) {
      const float gxl = w.st[st_lm(ly, l)] - ax, gyl = w.st[st_lm(ly, l) + 1] - ay;
      mloc[2 * l] = ca * gxl + sa * gyl;
      mloc[2 * l + 1] = -sa * gxl + ca * gyl;
    }
    tm.sync();
    // With more than one warp per environment the two passes run concurrently on the two halves of the
    // team (they write disjoint entries of H and b).
    const int halfA = TEAM == 32 ? TEAM : TEAM / 2;
    const bool doA = TEAM == 32 || lane < halfA, doB = TEAM == 32 || lane >= halfA;
    const int laneB = TEAM == 32 ? lane : lane - halfA;
    // ---- pass A: lane = pose slot k >= 1
    for (int k = doA ? 1 + lane : c; k < c; k += halfA) {
      uint64_t m = (uint64_t)w.rbm[k * ly.nw];
      if (ly.nw > 1) m |= (uint64_t)w.rbm[k * ly.nw + 1] << 32;
      if (!m) continue;
      const int r = ring_of(k, head, W), op = off_slot(ly, od, k, c);
      const float px = w.st[st_pose(k)], py = w.st[st_pose(k) + 1], pt = w.st[st_pose(k) + 2];
      float R[18];
#pragma unroll
      for (int t = 0; t < 18; ++t) R[t] = 0.f;
      int lnext = __ffsll((long long)m) - 1;  // measurements are prefetched one landmark ahead (they come from L2)
      float zr_n = rec[ly.o_zrb + (r * 2 + 0) * L + lnext], zb_n = rec[ly.o_zrb + (r * 2 + 1) * L + lnext];
      while (m) {
        const int l = lnext;
        const float zr = zr_n, zb = zb_n;
        m &= m - 1;
        if (m) {
          lnext = __ffsll((long long)m) - 1;
          zr_n = rec[ly.o_zrb + (r * 2 + 0) * L + lnext]; zb_n = rec[ly.o_zrb + (r * 2 + 1) * L + lnext];
        }
        const float mx = mloc[2 * l], my = mloc[2 * l + 1];
        const float dx = mx - px, dy = my - py;
        const float q = dx * dx + dy * dy, irho = rsqrt_fast(q), rho = q * irho, iq = irho * irho;
        const float r0 = rho - zr, r1 = wrapf(atan2_fast(dy, dx) - pt - zb);
        const float ux = dx * irho, uy = dy * irho, vx = -dy * iq, vy = dx * iq;     // J_l rows
        const float Ux = ca * ux - sa * uy, Uy = sa * ux + ca * uy;                  // J_g rows
        const float Vx = ca * vx - sa * vy, Vy = sa * vx + ca * vy;
        const float j0 = ux * my - uy * mx, j1 = vx * my - vy * mx;                  // J_a theta column
        const float wg0a = w0 * Ux, wg0b = w1 * Vx, wg1a = w0 * Uy, wg1b = w1 * Vy, wa2a = w0 * j0, wa2b = w1 * j1;
        // cross block <g_i, e_j>, pose columns e0 = (-ux,-vx), e1 = (-uy,-vy), e2 = (0,-1)
        const float ge00 = -(wg0a * ux + wg0b * vx), ge01 = -(wg0a * uy + wg0b * vy), ge02 = -wg0b;
        const float ge10 = -(wg1a * ux + wg1b * vx), ge11 = -(wg1a * uy + wg1b * vy), ge12 = -wg1b;
        const int ol = off_lm(ly, od, l);
        if (op < ol) {  // chain pose: landmark rows, pose columns
          float* r0p = w.H + rb_of(w, ol);
          float* r1p = w.H + rb_of(w, ol + 1);
          r0p[op] += ge00; r0p[op + 1] += ge01; r0p[op + 2] += ge02;
          r1p[op] += ge10; r1p[op + 1] += ge11; r1p[op + 2] += ge12;
        } else {        // newest pose: pose rows, landmark columns
          w.H[rb_of(w, op) + ol] += ge00; w.H[rb_of(w, op) + ol + 1] += ge10;
          w.H[rb_of(w, op + 1) + ol] += ge01; w.H[rb_of(w, op + 1) + ol + 1] += ge11;
          w.H[rb_of(w, op + 2) + ol] += ge02; w.H[rb_of(w, op + 2) + ol + 1] += ge12;
        }
        const float e0a = w0 * ux, e0b = w1 * vx, e1a = w0 * uy, e1b = w1 * vy;
        R[0] += e0a * ux + e0b * vx; R[1] += e1a * ux + e1b * vx; R[2] += e1a * uy + e1b * vy;
        R[3] += e0b; R[4] += e1b; R[5] += w1;
        R[6] -= e0a * r0 + e0b * r1; R[7] -= e1a * r0 + e1b * r1; R[8] -= w1 * r1;
        R[9] -= ge00; R[10] -= ge01; R[11] -= ge02;
        R[12] -= ge10; R[13] -= ge11; R[14] -= ge12;
        R[15] -= wa2a * ux + wa2b * vx; R[16] -= wa2a * uy + wa2b * vy; R[17] -= wa2b;
      }
      float* q0 = w.H + rb_of(w, op);
      float* q1 = w.H + rb_of(w, op + 1);
      float* q2 = w.H + rb_of(w, op + 2);
      q0[op] += R[0]; q1[op] += R[1]; q1[op + 1] += R[2];
      q2[op] += R[3]; q2[op + 1] += R[4]; q2[op + 2] += R[5];
      rhs[op] -= R[6]; rhs[op + 1] -= R[7]; rhs[op + 2] -= R[8];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        float* qa = w.H + rb_of(w, oA + i);
        qa[op] += R[9 + 3 * i]; qa[op + 1] += R[10 + 3 * i]; qa[op + 2] += R[11 + 3 * i];
      }
    }
    if (TEAM == 32) tm.sync();
    // ---- pass B: one landmark per group of 2^g lanes, which split its observing poses round-robin and
    // combine by shuffles (g > 0 when few landmarks are in view, else one lane would walk the whole window)
    float A[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};  // gg(3), <a2,g0>, <a2,g1>, <a2,a2>, <g0,r>, <g1,r>, <a2,r>
    const int nobs = __popcll(od.obs);
    int g = 0;
    while (g < 3 && (nobs << (g + 1)) <= 32) ++g;
    const int sub = laneB & ((1 << g) - 1), per = halfA >> g;
    for (int i0 = doB ? 0 : nobs; i0 < nobs; i0 += per) {
      const int idx = i0 + (laneB >> g);
      const bool inl = idx < nobs;
      const int l = inl ? nth_set_bit(od.obs, idx) : 0;
      const float mx = inl ? mloc[2 * l] : 0.f, my = inl ? mloc[2 * l + 1] : 0.f;
      float Lxx = 0.f, Lxy = 0.f, Lyy = 0.f, bgx = 0.f, bgy = 0.f, ag0 = 0.f, ag1 = 0.f, a22 = 0.f, a2r = 0.f;
      uint64_t km = 0ull;  // slots that observe this landmark
      if (inl)
        for (int k = 0; k < c; ++k) km |= (uint64_t)((w.rbm[k * ly.nw + (l >> 5)] >> (l & 31)) & 1u) << k;
      for (int j = 0; j < sub && km; ++j) km &= km - 1;  // this lane takes the bits sub, sub + 2^g, ...
      int knext = km ? __ffsll((long long)km) - 1 : 0;  // measurements prefetched one slot ahead (L2)
      int rn = ring_of(knext, head, W);
      float zr_n = km ? rec[ly.o_zrb + (rn * 2 + 0) * L + l] : 0.f, zb_n = km ? rec[ly.o_zrb + (rn * 2 + 1) * L + l] : 0.f;
      while (km) {
        const int k = knext;
        const float zr = zr_n, zb = zb_n;
        for (int j = 0; j < (1 << g) && km; ++j) km &= km - 1;
        if (km) {
          knext = __ffsll((long long)km) - 1;
          rn = ring_of(knext, head, W);
          zr_n = rec[ly.o_zrb + (rn * 2 + 0) * L + l]; zb_n = rec[ly.o_zrb + (rn * 2 + 1) * L + l];
        }
        const float* p = w.st + st_pose(k);
        const float dx = mx - p[0], dy = my - p[1];
        const float q = dx * dx + dy * dy, irho = rsqrt_fast(q), rho = q * irho, iq = irho * irho;
        const float r0 = rho - zr, r1 = wrapf(atan2_fast(dy, dx) - p[2] - zb);
        const float ux = dx * irho, uy = dy * irho, vx = -dy * iq, vy = dx * iq;
        const float Ux = ca * ux - sa * uy, Uy = sa * ux + ca * uy, Vx = ca * vx - sa * vy, Vy = sa * vx + ca * vy;
        const float j0 = ux * my - uy * mx, j1 = vx * my - vy * mx;
        const float wg0a = w0 * Ux, wg0b = w1 * Vx, wg1a = w0 * Uy, wg1b = w1 * Vy, wa2a = w0 * j0, wa2b = w1 * j1;
        Lxx += wg0a * Ux + wg0b * Vx; Lxy += wg0a * Uy + wg0b * Vy; Lyy += wg1a * Uy + wg1b * Vy;
        ag0 += wa2a * Ux + wa2b * Vx; ag1 += wa2a * Uy + wa2b * Vy; a22 += wa2a * j0 + wa2b * j1;
        bgx += wg0a * r0 + wg0b * r1; bgy += wg1a * r0 + wg1b * r1; a2r += wa2a * r0 + wa2b * r1;
      }
      for (int o = (1 << g) >> 1; o > 0; o >>= 1) {  // (uniform trip count: every lane of the warp is here)
        Lxx += __shfl_xor_sync(FULLMASK, Lxx, o); Lxy += __shfl_xor_sync(FULLMASK, Lxy, o); Lyy += __shfl_xor_sync(FULLMASK, Lyy, o);
        ag0 += __shfl_xor_sync(FULLMASK, ag0, o); ag1 += __shfl_xor_sync(FULLMASK, ag1, o); a22 += __shfl_xor_sync(FULLMASK, a22, o);
        bgx += __shfl_xor_sync(FULLMASK, bgx, o); bgy += __shfl_xor_sync(FULLMASK, bgy, o); a2r += __shfl_xor_sync(FULLMASK, a2r, o);
      }
      if (inl && sub == 0) {
        const int ol = off_lm(ly, od, l);
        float* r0p = w.H + rb_of(w, ol);
        float* r1p = w.H + rb_of(w, ol + 1);
        r0p[ol] += Lxx; r1p[ol] += Lxy; r1p[ol + 1] += Lyy;
        rhs[ol] -= bgx; rhs[ol + 1] -= bgy;
        // anchor rows x landmark columns: a0 = -g0, a1 = -g1, a2
        float* qa0 = w.H + rb_of(w, oA);
        float* qa1 = w.H + rb_of(w, oA + 1);
        float* qa2 = w.H + rb_of(w, oA + 2);
        qa0[ol] -= Lxx; qa0[ol + 1] -= Lxy;
        qa1[ol] -= Lxy; qa1[ol + 1] -= Lyy;
        qa2[ol] += ag0; qa2[ol + 1] += ag1;
        A[0] += Lxx; A[1] += Lxy; A[2] += Lyy; A[3] += ag0; A[4] += ag1; A[5] += a22;
        A[6] += bgx; A[7] += bgy; A[8] += a2r;
      }
    }
    tm.sync();
    tm.sum_n(A, lane);
    if (lane == 0) {  // anchor diagonal block and gradient
      float* qa0 = w.H + rb_of(w, oA);
      float* qa1 = w.H + rb_of(w, oA + 1);
      float* qa2 = w.H + rb_of(w, oA + 2);
      qa0[oA] += A[0]; qa1[oA] += A[1]; qa1[oA + 1] += A[2];
      qa2[oA] -= A[3]; qa2[oA + 1] -= A[4]; qa2[oA + 2] += A[5];
      rhs[oA] += A[6]; rhs[oA + 1] += A[7]; rhs[oA + 2] -= A[8];
    }
    tm.sync();
  }
}

// ------------------------------------------------------------------ S3: envelope Cholesky + solves
// Left-looking by 4-column blocks.  For block column J every lane owns a PAIR of rows below it (lane q
// of pass p: rows 4J + 2(q + 32p), +1) and accumulates its 2x4 strip S = H - sum_K L(i,K) L(J,K)' with
// 128-bit shared-memory loads (own rows: 2 loads, the four rows of block J: 4 broadcast loads, 32 FMA).
// The 4x4 diagonal tile (lanes 0 and 1 of pass 0) is shuffled to every lane, factorised redundantly in
// registers, and each lane finishes its rows by a 4-term forward substitution.  Diagonal slots store
// 1/L_jj.  Row np (rhs b; its pair twin np+1 is the same storage) rides along, so on exit it holds y = L^{-1} b.
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
#define FMA4(ACC, XV, BV)                                                                    \
  ACC = fmaf(-XV.x, BV.x, ACC); ACC = fmaf(-XV.y, BV.y, ACC); ACC = fmaf(-XV.z, BV.z, ACC); \
  ACC = fmaf(-XV.w, BV.w, ACC);

template <int TEAM, bool PAIRS, bool CACHE>
__device__ int cholesky(const Layout& ly, const WS& w, const Team<TEAM>& tm, int lane, int ncb, float rhi) {
  // ncb: number of leading column blocks whose factor is still valid from the previous factorisation of
  // this call (see assemble): there only the rhs pair -- the last entry of the column's list -- is
  // processed, on the lanes and with the K-split it has in a full pass, so y is bit-identical.
  const int np = ly.np, G = np >> 2;
  const Tables tb = tables_of(ly, w);
  constexpr int KUNROLL = SLAM_KUNROLL;
  int flag = 0;
  // Conditioning watch: the anchor's pivots are what fp32 loses first -- a robot that
  // dead-reckoned and re-observes a landmark has information on `a` spanning six decades.  Keep the assembled
  // diagonal of the three anchor rows; after the last column block compare it with the pivots.
  float ha0 = 0.f, ha1 = 0.f, ha2 = 0.f;
  if (rhi > 0.f) {   // rhi: this environment's threshold (slam_step_kernel), 0 = no watch
    const int oA = np - 3;
    ha0 = w.H[rb_of(w, oA) + oA]; ha1 = w.H[rb_of(w, oA + 1) + oA + 1]; ha2 = w.H[rb_of(w, oA + 2) + oA + 2];
  }
  for (int J = 0; J < G; ++J) {
    const int c0 = 4 * J;
    // the block's rows: pair A = rows c0, c0+1 (columns from fA), pair B = rows c0+2, c0+3 (from fB)
    // (!PAIRS: the four rows share first and length, one table entry describes them)
    const uint32_t hd = tb.hdr[J], eA = tb.ptab[2 * J], eB = PAIRS ? tb.ptab[2 * J + 1] : 0u;
    const int fA = (int)((eA >> 14) & 0x7fu) << 2, lenA = (int)(eA >> 21) << 2;
    const int fB = PAIRS ? (int)((eB >> 14) & 0x7fu) << 2 : fA;
    const float* rJ0 = w.H + ((int)(eA & 0x3fffu) << 2) - fA;
    const float* rJ1 = rJ0 + lenA;
    const float* rJ2 = PAIRS ? w.H + ((int)(eB & 0x3fffu) << 2) - fB : rJ1 + lenA;
    const float* rJ3 = rJ2 + (PAIRS ? (int)(eB >> 21) << 2 : lenA);
    const int fJ = min(fA, fB), fH = max(fA, fB);    // both pairs have entries from fH on, one of them from fJ
    // The ACTIVE row pairs of this column (compact list from the symbolic phase) sit on the lowest
    // threads.  K-split: when fewer pairs than threads, `ch` adjacent lanes share one pair and
    // split the dot-product range; partial sums are combined by shuffles.
    const unsigned char* alist = tb.alist + (hd & 0x3fffu);
    const int cnt = (int)((hd >> 14) & 0xffu);
    const int lg = (int)((hd >> (TEAM == 32 ? 22 : (TEAM == 64 ? 24 : 26))) & 3u);
    const int ch = 1 << lg;
    const int per_pass = TEAM >> lg;
    const int t = lane & (ch - 1);
    float d0 = 1.f, d1 = 1.f, d2 = 1.f, d3 = 1.f, l10 = 0.f, l20 = 0.f, l21 = 0.f, l30 = 0.f, l31 = 0.f, l32 = 0.f;
    const bool cached = CACHE && J < ncb;   // (CACHE = windows with landmarks: pose-only kernels drop the path)
    if (cached) {
      const float4 t0 = ld4(rJ0 + c0), t1 = ld4(rJ1 + c0), t2 = ld4(rJ2 + c0), t3 = ld4(rJ3 + c0);
      d0 = t0.x; l10 = t1.x; d1 = t1.y; l20 = t2.x; l21 = t2.y; d2 = t2.z; l30 = t3.x; l31 = t3.y; l32 = t3.z; d3 = t3.w;
    }
    for (int q0 = cached ? ((cnt - 1) & ~(per_pass - 1)) : 0; q0 < cnt; q0 += per_pass) {
      const bool first_pass = !cached && q0 == 0;
      const int q = q0 + (lane >> lg);
      const bool act = cached ? q == cnt - 1 : q < cnt;
      // a warp without any pair in this pass only takes part in the barriers
      const bool warp_idle = TEAM > 32 && q0 + ((lane & ~31) >> lg) >= cnt;
      if (warp_idle) {
        if (first_pass) tm.sync();
        continue;
      }
      float4 a0 = make_float4(0.f, 0.f, 0.f, 0.f), a1 = a0;
      float* p0 = nullptr;
      float* p1 = nullptr;
      if (act) {
        const uint32_t e = tb.ptab[alist[q]];
        const int fi = (int)((e >> 14) & 0x7fu) << 2;
        p0 = w.H + ((int)(e & 0x3fffu) << 2) - fi;
        p1 = p0 + ((int)(e >> 21) << 2);
        if (t == 0) { a0 = ld4(p0 + c0); a1 = ld4(p1 + c0); }  // (rows np, np+1 are the rhs pair)
        const int ks = max(fi, fJ);
        const int nblk = (c0 - ks) >> 2;
        const int kb = ks + 4 * ((t * nblk) >> lg), ke = ks + 4 * (((t + 1) * nblk) >> lg);
        if (PAIRS && fA != fB) {  // (block-uniform) columns [kb, fH): only the earlier pair of the block has entries
          const float* rL0 = fA < fB ? rJ0 : rJ2;
          const float* rL1 = fA < fB ? rJ1 : rJ3;
          float u00 = 0.f, u01 = 0.f, u10 = 0.f, u11 = 0.f;
          const int km = min(ke, fH);
          for (int k = kb; k < km; k += 4) {
            const float4 x0 = ld4(p0 + k), x1 = ld4(p1 + k);
            const float4 b0 = ld4(rL0 + k), b1 = ld4(rL1 + k);
            FMA4(u00, x0, b0) FMA4(u01, x0, b1) FMA4(u10, x1, b0) FMA4(u11, x1, b1)
          }
          if (fA < fB) { a0.x += u00; a0.y += u01; a1.x += u10; a1.y += u11; }
          else { a0.z += u00; a0.w += u01; a1.z += u10; a1.w += u11; }
        }
#pragma unroll KUNROLL
        for (int k = max(kb, fH); k < ke; k += 4) {
          const float4 x0 = ld4(p0 + k), x1 = ld4(p1 + k);
          const float4 b0 = ld4(rJ0 + k), b1 = ld4(rJ1 + k), b2 = ld4(rJ2 + k), b3 = ld4(rJ3 + k);
          FMA4(a0.x, x0, b0) FMA4(a0.y, x0, b1) FMA4(a0.z, x0, b2) FMA4(a0.w, x0, b3)
          FMA4(a1.x, x1, b0) FMA4(a1.y, x1, b1) FMA4(a1.z, x1, b2) FMA4(a1.w, x1, b3)
        }
      }
      for (int o = ch >> 1; o > 0; o >>= 1) {  // combine the K-split partial sums (uniform trip count)
        a0.x += __shfl_xor_sync(FULLMASK, a0.x, o); a0.y += __shfl_xor_sync(FULLMASK, a0.y, o);
        a0.z += __shfl_xor_sync(FULLMASK, a0.z, o); a0.w += __shfl_xor_sync(FULLMASK, a0.w, o);
        a1.x += __shfl_xor_sync(FULLMASK, a1.x, o); a1.y += __shfl_xor_sync(FULLMASK, a1.y, o);
        a1.z += __shfl_xor_sync(FULLMASK, a1.z, o); a1.w += __shfl_xor_sync(FULLMASK, a1.w, o);
      }
      if (first_pass) {  // diagonal tile: thread 0 holds rows c0, c0+1; thread `ch` rows c0+2, c0+3
        float s00, s10, s11, s20, s21, s22, s30, s31, s32, s33;
        if (TEAM == 32) {
          s00 = __shfl_sync(FULLMASK, a0.x, 0);
          s10 = __shfl_sync(FULLMASK, a1.x, 0); s11 = __shfl_sync(FULLMASK, a1.y, 0);
          s20 = __shfl_sync(FULLMASK, a0.x, ch); s21 = __shfl_sync(FULLMASK, a0.y, ch); s22 = __shfl_sync(FULLMASK, a0.z, ch);
          s30 = __shfl_sync(FULLMASK, a1.x, ch); s31 = __shfl_sync(FULLMASK, a1.y, ch); s32 = __shfl_sync(FULLMASK, a1.z, ch);
          s33 = __shfl_sync(FULLMASK, a1.w, ch);
        } else {
          float* dg = tm.scr + 16;
          if (lane == 0) { dg[0] = a0.x; dg[1] = a1.x; dg[2] = a1.y; }
          if (lane == ch) { dg[3] = a0.x; dg[4] = a0.y; dg[5] = a0.z; dg[6] = a1.x; dg[7] = a1.y; dg[8] = a1.z; dg[9] = a1.w; }
          tm.sync();
          s00 = dg[0]; s10 = dg[1]; s11 = dg[2]; s20 = dg[3]; s21 = dg[4]; s22 = dg[5];
          s30 = dg[6]; s31 = dg[7]; s32 = dg[8]; s33 = dg[9];
        }
        bool bad = !(s00 > 0.f);
        d0 = rsqrt_fast(s00);
        l10 = s10 * d0; l20 = s20 * d0; l30 = s30 * d0;
        const float t11 = fmaf(-l10, l10, s11);
        bad |= !(t11 > 0.f);
        d1 = rsqrt_fast(t11);
        l21 = fmaf(-l20, l10, s21) * d1; l31 = fmaf(-l30, l10, s31) * d1;
        const float t22 = fmaf(-l21, l21, fmaf(-l20, l20, s22));
        bad |= !(t22 > 0.f);
        d2 = rsqrt_fast(t22);
        l32 = fmaf(-l31, l21, fmaf(-l30, l20, s32)) * d2;
        const float t33 = fmaf(-l32, l32, fmaf(-l31, l31, fmaf(-l30, l30, s33)));
        bad |= !(t33 > 0.f);
        d3 = rsqrt_fast(t33);
        if (bad) {
          flag |= ENV_NOT_PD;
          if (!(s00 > 0.f)) d0 = 1.f;
          if (!(t11 > 0.f)) d1 = 1.f;
          if (!(t22 > 0.f)) d2 = 1.f;
          if (!(t33 > 0.f)) d3 = 1.f;
        }
        // rows np-3 .. np-1 of the last block are the anchor: H_ii / L_ii^2 = H_ii d_i^2
        if (J == G - 1 && fmaxf(fmaxf(ha0 * d1 * d1, ha1 * d2 * d2), ha2 * d3 * d3) > rhi && rhi > 0.f) flag |= ENV_ILLCOND;
      }
      if (act && t == 0) {
        if (first_pass && q < 2) {
          if (q == 0) { a0 = make_float4(d0, 0.f, 0.f, 0.f); a1 = make_float4(l10, d1, 0.f, 0.f); }
          else { a0 = make_float4(l20, l21, d2, 0.f); a1 = make_float4(l30, l31, l32, d3); }
        } else {
          a0.x *= d0; a0.y = fmaf(-a0.x, l10, a0.y) * d1;
          a0.z = fmaf(-a0.y, l21, fmaf(-a0.x, l20, a0.z)) * d2;
          a0.w = fmaf(-a0.z, l32, fmaf(-a0.y, l31, fmaf(-a0.x, l30, a0.w))) * d3;
          a1.x *= d0; a1.y = fmaf(-a1.x, l10, a1.y) * d1;
          a1.z = fmaf(-a1.y, l21, fmaf(-a1.x, l20, a1.z)) * d2;
          a1.w = fmaf(-a1.z, l32, fmaf(-a1.y, l31, fmaf(-a1.x, l30, a1.w))) * d3;
        }
        st4(p0 + c0, a0);
        st4(p1 + c0, a1);
      }
    }
    tm.sync();
  }
  return flag;
}

// Solves L' delta = y in place in row np, by 4-row blocks from the bottom: delta_I from the diagonal
// tile (every lane redundantly), then y_K -= L(I,K)' delta_I with lanes over the column blocks K.
template <int TEAM, bool PAIRS>
__device__ void back_substitute(const Layout& ly, const WS& w, const Team<TEAM>& tm, int lane) {
  const int np = ly.np, G = np >> 2;
  const Tables tb = tables_of(ly, w);
  float* y = w.H + rb_of(w, np);
  for (int I = G - 1; I >= 0; --I) {
    const int c0 = 4 * I;
    const uint32_t eA = tb.ptab[2 * I], eB = PAIRS ? tb.ptab[2 * I + 1] : 0u;
    const int fA = (int)((eA >> 14) & 0x7fu) << 2, lenA = (int)(eA >> 21) << 2;
    const int fB = PAIRS ? (int)((eB >> 14) & 0x7fu) << 2 : fA, fI = min(fA, fB);
    const float* r0 = w.H + ((int)(eA & 0x3fffu) << 2) - fA;
    const float* r1 = r0 + lenA;
    const float* r2 = PAIRS ? w.H + ((int)(eB & 0x3fffu) << 2) - fB : r1 + lenA;
    const float* r3 = r2 + (PAIRS ? (int)(eB >> 21) << 2 : lenA);
    const float4 yy = ld4(y + c0), t0 = ld4(r0 + c0), t1 = ld4(r1 + c0), t2 = ld4(r2 + c0), t3 = ld4(r3 + c0);
    const float e3 = yy.w * t3.w;
    const float e2 = fmaf(-t3.z, e3, yy.z) * t2.z;
    const float e1 = fmaf(-t3.y, e3, fmaf(-t2.y, e2, yy.y)) * t1.y;
    const float e0 = fmaf(-t3.x, e3, fmaf(-t2.x, e2, fmaf(-t1.x, e1, yy.x))) * t0.x;
    tm.sync();
    if (lane == 0) st4(y + c0, make_float4(e0, e1, e2, e3));
    for (int k = fI + 4 * lane; k < c0; k += 4 * TEAM) {
      float4 v = ld4(y + k);
      if (!PAIRS || k >= fA) {   // (a pair has no entries left of its first column)
        const float4 x0 = ld4(r0 + k), x1 = ld4(r1 + k);
        v.x = fmaf(-x1.x, e1, fmaf(-x0.x, e0, v.x)); v.y = fmaf(-x1.y, e1, fmaf(-x0.y, e0, v.y));
        v.z = fmaf(-x1.z, e1, fmaf(-x0.z, e0, v.z)); v.w = fmaf(-x1.w, e1, fmaf(-x0.w, e0, v.w));
      }
      if (!PAIRS || k >= fB) {
        const float4 x2 = ld4(r2 + k), x3 = ld4(r3 + k);
        v.x = fmaf(-x3.x, e3, fmaf(-x2.x, e2, v.x)); v.y = fmaf(-x3.y, e3, fmaf(-x2.y, e2, v.y));
        v.z = fmaf(-x3.z, e3, fmaf(-x2.z, e2, v.z)); v.w = fmaf(-x3.w, e3, fmaf(-x2.w, e2, v.w));
      }
      st4(y + k, v);
    }
    tm.sync();
  }
}

// v <- v + delta (R1: additive, angles wrapped).  Returns ENV_NONFINITE if the update is not finite.
template <int TEAM>
__device__ int apply_update(const Layout& ly, const Ord& od, const WS& w, const Team<TEAM>& tm, int lane, int c, const Masks& mk) {
  const int W = ly.W, L = ly.L;
  const float* dl = w.H + rb_of(w, ly.np);
  int bad = 0;
  if (lane < 3) {
    const float d = dl[off_a(ly) + lane];
    bad |= !isfinite(d);
    const float v = w.st[lane] + d;
    w.st[lane] = lane == 2 ? wrapf(v) : v;
  }
  for (int i = lane; i < 3 * (c - 1); i += TEAM) {
    const int k = 1 + i / 3, j = i - 3 * (k - 1);
    const float d = dl[off_slot(ly, od, k, c) + j];
    bad |= !isfinite(d);
    const float v = w.st[st_pose(k) + j] + d;
    w.st[st_pose(k) + j] = j == 2 ? wrapf(v) : v;
  }
  for (int i = lane; i < 2 * L; i += TEAM) {
    if (!((mk.act >> (i >> 1)) & 1ull)) continue;
    const float d = dl[off_lm(ly, od, i >> 1) + (i & 1)];
    bad |= !isfinite(d);
    w.st[3 + 3 * W + i] += d;
  }
  const bool anybad = tm.any(bad != 0, lane);
  tm.sync();
  return anybad ? ENV_NONFINITE : 0;
}

// ------------------------------------------------------------------ S4: covariance of the newest pose
// Sigma_6 = (L_t L_t')^{-1} from the trailing 6x6 of L (variables: newest pose e, anchor a), then
// Sigma_t = J Sigma_6 J' with x = a (+) e (A.4).  O(1) per environment, done in fp64 by lane 0.
template <int TEAM>
__device__ void covariance(const Layout& ly, const WS& w, const Team<TEAM>& tm, int lane, int env, int c, const StepIO& io) {
  if (lane >= 32) return;  // first warp of the team; stages separated by __syncwarp, fp64 scratch in shared memory
  const int n = ly.np, N = ly.N;
  // fp64 scratch (135 doubles) at the start of this environment's pool share: the factor is dead after
  // this call, and the trailing block is read into registers before the first scratch word is written
  double* Lm = reinterpret_cast<double*>(w.H);          // [6][6] trailing block of L (diagonal = 1/L_jj)
  double* Li = Lm + 36;                                 // [6][6] its inverse
  double* S6 = Li + 36;                                 // [6][6] Sigma_6 = Li' Li
  double* T = S6 + 36;                                  // [6][3] Sigma_6 J'
  double* S = T + 18;                                   // [3][3] Sigma_t
  // J = [J_e | J_a], J_e = blockdiag(Rot(a_th), 1), J_a = [[1,0,-dy],[0,1,dx],[0,0,1]], d = Rot(a_th) t_e.
  // With a single pose (c == 1) the newest-pose block is an identity placeholder: J_e = 0, J_a = I.
  float saf, caf;
  sincos_pi(w.st[2], &saf, &caf);
  const double ca = (double)caf, sa = (double)saf, je = c >= 2 ? 1.0 : 0.0;
  const float* e = w.st + st_pose(c >= 2 ? c - 1 : 0);
  const double dx = ca * e[0] - sa * e[1], dy = sa * e[0] + ca * e[1];
  const double J[3][6] = {{je * ca, -je * sa, 0, 1, 0, -dy}, {je * sa, je * ca, 0, 0, 1, dx}, {0, 0, je, 0, 0, 1}};
  float lrow[6];
  if (lane < 6) {  // row `lane` of the trailing block
    const int i = n - 6 + lane, fi = first_of(w, i);
#pragma unroll
    for (int y = 0; y < 6; ++y) {
      const int j = n - 6 + y;
      float v = 0.f;
      if (y == lane) v = w.H[rb_of(w, i) + i];
      else if (y < lane && j >= fi) v = w.H[rb_of(w, i) + j];
      lrow[y] = v;
    }
  }
  __syncwarp();
  if (lane < 6) {
#pragma unroll
    for (int y = 0; y < 6; ++y) { Lm[lane * 6 + y] = (double)lrow[y]; Li[lane * 6 + y] = 0.0; }
  }
  __syncwarp();
  if (lane < 6) {  // column `lane` of L^{-1} by forward substitution
    const int col = lane;
    for (int x = col; x < 6; ++x) {
      double sum = (x == col) ? 1.0 : 0.0;
      for (int k = col; k < x; ++k) sum -= Lm[x * 6 + k] * Li[k * 6 + col];
      Li[x * 6 + col] = sum * Lm[x * 6 + x];
    }
  }
  __syncwarp();
  if (lane < 6) {  // row `lane` of Sigma_6 = Li' Li
    for (int y = 0; y < 6; ++y) {
      double sum = 0.0;
      for (int k = (lane > y ? lane : y); k < 6; ++k) sum += Li[k * 6 + lane] * Li[k * 6 + y];
      S6[lane * 6 + y] = sum;
    }
  }
  __syncwarp();
  if (lane < 6) {  // row `lane` of T = Sigma_6 J'
    for (int j = 0; j < 3; ++j) {
      double sum = 0.0;
      for (int q = 0; q < 6; ++q) sum += S6[lane * 6 + q] * J[j][q];
      T[lane * 3 + j] = sum;
    }
  }
  __syncwarp();
  if (lane < 9) {  // Sigma_t = J T
    const int x = lane / 3, y = lane - 3 * x;
    double sum = 0.0;
    for (int p2 = 0; p2 < 6; ++p2) sum += J[x][p2] * T[p2 * 3 + y];
    S[lane] = sum;
  }
  __syncwarp();
  if (lane < 9) {  // R20: symmetrise; outputs
    const int x = lane / 3, y = lane - 3 * x;
    const float v = (float)(0.5 * (S[x * 3 + y] + S[y * 3 + x]));
    io.cov_cache[(size_t)lane * N + env] = v;
    if (io.cov) io.cov[(size_t)lane * N + env] = v;
  }
  if (lane == 0) {
    const double s01 = 0.5 * (S[1] + S[3]), s02 = 0.5 * (S[2] + S[6]), s12 = 0.5 * (S[5] + S[7]);
    const double det = S[0] * (S[4] * S[8] - s12 * s12) - s01 * (s01 * S[8] - s12 * s02) + s02 * (s01 * s12 - S[4] * s02);
    const float ld = logf((float)det);
    io.cov_cache[(size_t)9 * N + env] = ld;
    if (io.logdet) io.logdet[env] = ld;
    if (io.dopt) io.dopt[env] = expf(ld * (1.0f / 3.0f));
  }
  __syncwarp();
}

// ------------------------------------------------------------------ S5: marginalise the oldest pose
// Works on the SUPPORT of the sub-problem only (old prior + factors touching slot 0), dimension s:
//   H_s, gamma_s  ->  congruence with N = dv/du = E + X P_w'  (E block diagonal, X the w-column)
//   ->  Schur complement over w = e_1  ->  (Lambda', g', vbar') on the support without w.
// Block order of the support: [a | pose slots ascending (slot 1 = w first) | landmarks ascending].
struct Etype { float p, q, u, v; };  // E = [[p,-q,u],[q,p,v],[0,0,1]]

__device__ __forceinline__ int tri(int i, int j) { return (i * (i + 1) >> 1) + j; }  // i >= j
__device__ __forceinline__ float sym_get(const float* Hs, int i, int j) { return i >= j ? Hs[tri(i, j)] : Hs[tri(j, i)]; }

// Shared-memory words the marginalisation of this environment needs (support of the sub-problem).
__device__ __forceinline__ int marg_need(const Layout& ly, const WS& w, int lane, int c, const Masks& mk) {
  uint64_t lc0 = 0ull;
  for (int base = 0; base < c; base += 32) {
    const int k = base + (lane & 31);
    const uint32_t bal = __ballot_sync(FULLMASK, k >= 1 && k < c && w.lct[k] == 0);
    lc0 |= (uint64_t)bal << base;
  }
  uint64_t rb0 = 0ull;
  if (ly.L > 0) { rb0 = (uint64_t)w.rbm[0]; if (ly.nw > 1) rb0 |= (uint64_t)w.rbm[1] << 32; }
  const int s = 3 + 3 * __popcll(mk.ps | 2ull | lc0) + 2 * __popcll(mk.ls | rb0);
  return (s * (s + 1) >> 1) + 8 * s;
}

template <int TEAM>
__device__ int marginalize(const Layout& ly, const Params& pr, float* rec, const WS& w, const Team<TEAM>& tm, int lane, int head, int c,
                           Masks& mk, int s_old) {
  const int W = ly.W, L = ly.L;
  int* reci = (int*)rec;
  uint32_t* recu = (uint32_t*)rec;
  // --- A. new support masks
  uint64_t lc0 = 0ull;
  for (int base = 0; base < c; base += 32) {  // every warp of the team builds the whole mask
    const int k = base + (lane & 31);
    const uint32_t bal = __ballot_sync(FULLMASK, k >= 1 && k < c && w.lct[k] == 0);
    lc0 |= (uint64_t)bal << base;
  }
  uint64_t rb0 = 0ull;
  if (L > 0) { rb0 = (uint64_t)w.rbm[0]; if (ly.nw > 1) rb0 |= (uint64_t)w.rbm[1] << 32; }
  const uint64_t nps = mk.ps | 2ull | lc0, nls = mk.ls | rb0;
  const int npn = __popcll(nps), nln = __popcll(nls);
  const int s = 3 + 3 * npn + 2 * nln, nbk = 1 + npn + nln;
  const int npo = __popcll(mk.ps);
  if ((s * (s + 1) >> 1) + 8 * s > ly.cap) return 4;  // cannot happen: the pool holds a dense window
  float* Hs = w.H;
  float* gam = Hs + (s * (s + 1) >> 1);
  float* X = gam + s;
  float* Q = X + 3 * s;
  int* omap = (int*)(Q + 3 * s);
  int* nidx = reinterpret_cast<int*>(w.sup);  // the old table is dead once step B has read it

  // --- B. old displacement d, old -> new scalar map, new state-index table
  for (int p = lane; p < s_old; p += TEAM) {
    const uint32_t e = w.sup[p];
    float d = w.st[sup_idx(e)] - rec[ly.o_vbar + p];
    if (sup_angle(e)) d = wrapf(d);
    w.sds[p] = d;
    int P;
    if (p < 3) P = p;
    else if (p < 3 + 3 * npo) {
      const int b = (p - 3) / 3, j = (p - 3) - 3 * b, k = nth_set_bit(mk.ps, b);
      P = 3 + 3 * __popcll(nps & lowmask(k)) + j;
    } else {
      const int q = p - 3 - 3 * npo, b = q >> 1, j = q & 1, l = nth_set_bit(mk.ls, b);
      P = 3 + 3 * npn + 2 * __popcll(nls & lowmask(l)) + j;
    }
    omap[p] = P;
  }
  for (int t = lane; t < (s * (s + 1) >> 1) + s; t += TEAM) Hs[t] = 0.f;  // Hs and gam
  tm.sync();
  const float a_th = w.st[2];
  float sa, ca;
  sincos_pi(a_th, &sa, &ca);
  const float x1 = w.st[st_pose(1)], y1 = w.st[st_pose(1) + 1], th1 = w.st[st_pose(1) + 2];
  float s1, c1;
  sincos_pi(th1, &s1, &c1);
  const float ddx = ca * x1 - sa * y1, ddy = sa * x1 + ca * y1;  // d = Rot(a_th) t_1
  // new tables + X rows (step E)
  for (int p = lane; p < s; p += TEAM) {
    int id;
    float X0, X1, X2;
    if (p < 3) {
      id = p | (p == 2 ? 0x10000 : 0);
      // B = da/dw = [[-ca, sa, -dy], [-sa, -ca, dx], [0, 0, -1]]
      X0 = p == 0 ? -ca : (p == 1 ? -sa : 0.f);
      X1 = p == 0 ? sa : (p == 1 ? -ca : 0.f);
      X2 = p == 0 ? -ddy : (p == 1 ? ddx : -1.f);
    } else if (p < 3 + 3 * npn) {
      const int b = (p - 3) / 3, j = (p - 3) - 3 * b, k = nth_set_bit(nps, b);
      id = (st_pose(k) + j) | (j == 2 ? 0x10000 : 0);
      if (k == 1) { X0 = 0.f; X1 = 0.f; X2 = 0.f; }
      else {  // C_k = de_k/dw = [[1,0,-(y_k-y_1)],[0,1,x_k-x_1],[0,0,1]]
        X0 = j == 0 ? 1.f : 0.f; X1 = j == 1 ? 1.f : 0.f;
        X2 = j == 0 ? -(w.st[st_pose(k) + 1] - y1) : (j == 1 ? (w.st[st_pose(k)] - x1) : 1.f);
      }
    } else {
      const int q = p - 3 - 3 * npn, b = q >> 1, j = q & 1, l = nth_set_bit(nls, b);
      id = st_lm(ly, l) + j;
      X0 = 0.f; X1 = 0.f; X2 = 0.f;  // landmarks are global: untouched by re-anchoring
    }
    nidx[p] = id;
    X[3 * p] = X0; X[3 * p + 1] = X1; X[3 * p + 2] = X2;
  }
  tm.sync();
  // --- C. scatter the old prior
  {
    const float* lam = rec + ly.o_lam;
    const int ntri = s_old * (s_old + 1) >> 1;
    int tp = tri_row(lane), tq = lane - (tp * (tp + 1) >> 1);
#pragma unroll 4
    for (int t = lane; t < ntri; t += TEAM) {
      Hs[tri(omap[tp], omap[tq])] = lam[t];
      tri_advance(tp, tq, TEAM);
    }
    for (int p = lane; p < s_old; p += TEAM) {
      float acc = rec[ly.o_g + p];
      const float* lrow = lam + (p * (p + 1) >> 1);
      for (int q = 0; q <= p; ++q) acc = fmaf(lrow[q], w.sds[q], acc);
      for (int q = p + 1; q < s_old; ++q) acc = fmaf(lam[(q * (q + 1) >> 1) + p], w.sds[q], acc);
      gam[omap[p]] = acc;
    }
  }
  tm.sync();
  // --- D. factors touching slot 0 (the frame): J_j = I for between factors
  if (lane < 3) {
    float r = w.st[st_pose(1) + lane] - rec[ly.o_zodo + 3 * ring_of(1, head, W) + lane];
    if (lane == 2) r = wrapf(r);
    Hs[tri(3 + lane, 3 + lane)] += pr.om_odo[lane];
    gam[3 + lane] += pr.om_odo[lane] * r;
  }
  tm.sync();
  for (int k = 1 + lane; k < c; k += TEAM) {
    if (w.lct[k] == 0) {
      const int P = 3 + 3 * __popcll(nps & lowmask(k));
      for (int x = 0; x < 3; ++x) {
        float r = w.st[st_pose(k) + x] - rec[ly.o_zlc + 3 * ring_of(k, head, W) + x];
        if (x == 2) r = wrapf(r);
        Hs[tri(P + x, P + x)] += pr.om_lc[x];
        gam[P + x] += pr.om_lc[x] * r;
      }
    }
  }
  if ((mk.um & 1ull) && lane == 0) {  // unary factor of slot 0 (x = a, J_a = I)
    const float* om = rec + ly.o_omun + 6 * head;
    const float r0 = w.st[0] - rec[ly.o_zun + 3 * head], r1 = w.st[1] - rec[ly.o_zun + 3 * head + 1];
    const float r2 = wrapf(w.st[2] - rec[ly.o_zun + 3 * head + 2]);
    Hs[tri(0, 0)] += om[0]; Hs[tri(1, 0)] += om[1]; Hs[tri(1, 1)] += om[2];
    Hs[tri(2, 0)] += om[3]; Hs[tri(2, 1)] += om[4]; Hs[tri(2, 2)] += om[5];
    gam[0] += om[0] * r0 + om[1] * r1 + om[3] * r2;
    gam[1] += om[1] * r0 + om[2] * r1 + om[4] * r2;
    gam[2] += om[3] * r0 + om[4] * r1 + om[5] * r2;
  }
  tm.sync();
  if (L > 0 && rb0) {  // range-bearing from slot 0 (observing pose x = a): blocks a and g
    float A[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int l = lane; l < L; l += TEAM) {
      if ((rb0 >> l) & 1ull) {
        const float zr = rec[ly.o_zrb + (head * 2 + 0) * L + l], zb = rec[ly.o_zrb + (head * 2 + 1) * L + l];
        const float gxl = w.st[st_lm(ly, l)] - w.st[0], gyl = w.st[st_lm(ly, l) + 1] - w.st[1];
        const float dx = ca * gxl + sa * gyl, dy = -sa * gxl + ca * gyl;  // m = Rot(a_th)'(g - a_t)
        const float q = dx * dx + dy * dy, irho = rsqrt_fast(q), rho = q * irho, iq = irho * irho;
        const float r0 = rho - zr, r1 = wrapf(atan2_fast(dy, dx) - zb);
        const float ux = dx * irho, uy = dy * irho, vx = -dy * iq, vy = dx * iq;
        const float Ux = ca * ux - sa * uy, Uy = sa * ux + ca * uy, Vx = ca * vx - sa * vy, Vy = sa * vx + ca * vy;
        const float j0 = ux * dy - uy * dx, j1 = vx * dy - vy * dx;       // = 0, -1 (kept in the general form)
        const float wg0a = pr.om_rb[0] * Ux, wg0b = pr.om_rb[1] * Vx, wg1a = pr.om_rb[0] * Uy, wg1b = pr.om_rb[1] * Vy;
        const float wa2a = pr.om_rb[0] * j0, wa2b = pr.om_rb[1] * j1;
        const float gg00 = wg0a * Ux + wg0b * Vx, gg01 = wg0a * Uy + wg0b * Vy, gg11 = wg1a * Uy + wg1b * Vy;
        const float a2g0 = wa2a * Ux + wa2b * Vx, a2g1 = wa2a * Uy + wa2b * Vy, a2a2 = wa2a * j0 + wa2b * j1;
        const float g0r = wg0a * r0 + wg0b * r1, g1r = wg1a * r0 + wg1b * r1, a2r = wa2a * r0 + wa2b * r1;
        const int P = 3 + 3 * npn + 2 * __popcll(nls & lowmask(l));
        Hs[tri(P, P)] += gg00; Hs[tri(P + 1, P)] += gg01; Hs[tri(P + 1, P + 1)] += gg11;
        gam[P] += g0r; gam[P + 1] += g1r;
        // landmark rows x anchor columns: <g_i, a_j>, a0 = -g0, a1 = -g1, a2 = (j0, j1)
        Hs[tri(P, 0)] -= gg00; Hs[tri(P, 1)] -= gg01; Hs[tri(P, 2)] += a2g0;
        Hs[tri(P + 1, 0)] -= gg01; Hs[tri(P + 1, 1)] -= gg11; Hs[tri(P + 1, 2)] += a2g1;
        A[0] += gg00; A[1] += gg01; A[2] += gg11; A[3] += a2g0; A[4] += a2g1; A[5] += a2a2;
        A[6] += g0r; A[7] += g1r; A[8] += a2r;
      }
    }
    tm.sum_n(A, lane);
    if (lane == 0) {
      Hs[tri(0, 0)] += A[0]; Hs[tri(1, 0)] += A[1]; Hs[tri(1, 1)] += A[2];
      Hs[tri(2, 0)] -= A[3]; Hs[tri(2, 1)] -= A[4]; Hs[tri(2, 2)] += A[5];
      gam[0] -= A[6]; gam[1] -= A[7]; gam[2] += A[8];
    }
  }
  tm.sync();
  // --- F. Q = H_s X;  Y = X'Q;  gx = X'gamma
  float Y[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, gx[3] = {0, 0, 0};
  for (int p = lane; p < s; p += TEAM) {
    float q0 = 0.f, q1 = 0.f, q2 = 0.f;
    {
      // the landmark rows of X are zero (landmarks are global: untouched by re-anchoring): only the anchor and
      // pose columns of H_s contribute (the skipped terms are exact zeros)
      const int sx = 3 + 3 * npn;
      for (int q = 0; q < sx; ++q) {
        const float h = sym_get(Hs, p, q);
        q0 = fmaf(h, X[3 * q], q0); q1 = fmaf(h, X[3 * q + 1], q1); q2 = fmaf(h, X[3 * q + 2], q2);
      }
      Q[3 * p] = q0; Q[3 * p + 1] = q1; Q[3 * p + 2] = q2;
      const float xa = X[3 * p], xb = X[3 * p + 1], xc = X[3 * p + 2], gp = gam[p];
      Y[0] += xa * q0; Y[1] += xa * q1; Y[2] += xa * q2;
      Y[3] += xb * q0; Y[4] += xb * q1; Y[5] += xb * q2;
      Y[6] += xc * q0; Y[7] += xc * q1; Y[8] += xc * q2;
      gx[0] += xa * gp; gx[1] += xb * gp; gx[2] += xc * gp;
    }
  }
  tm.sum_n(Y, lane);
  tm.sum_n(gx, lane);
  tm.sync();
  // --- G. G = E' H_s E block by block (in place);  T_b = E_b' Q_b;  gamma_b = E_b' gamma_b
  auto etype = [&](int b) -> Etype {
    if (b == 0) return Etype{1.f, 0.f, ddy, -ddx};          // A = da/da'
    if (b == 1 || b > npn) return Etype{1.f, 0.f, 0.f, 0.f};  // w and the (global) landmarks: identity
    return Etype{c1, s1, 0.f, 0.f};                           // blockdiag(Rot(th_1), 1)
  };
  auto bpos = [&](int b) -> int { return b == 0 ? 0 : (b <= npn ? 3 + 3 * (b - 1) : 3 + 3 * npn + 2 * (b - 1 - npn)); };
  const int npairs = nbk * (nbk + 1) >> 1;
  int bi = tri_row(lane), bj = lane - (bi * (bi + 1) >> 1);
  for (int t = lane; t < npairs; t += TEAM, tri_advance(bi, bj, TEAM)) {
    // E is the identity for w (block 1) and for the landmarks: a pair of such blocks keeps its entries as they are
    if ((bi == 1 || bi > npn) && (bj == 1 || bj > npn)) continue;
    const int pi = bpos(bi), pj = bpos(bj), di = bi <= npn ? 3 : 2, dj = bj <= npn ? 3 : 2;
    const Etype Ei = etype(bi), Ej = etype(bj);
    float M[3][3];
#pragma unroll
    for (int x = 0; x < 3; ++x)
#pragma unroll
      for (int y = 0; y < 3; ++y) M[x][y] = (x < di && y < dj) ? sym_get(Hs, pi + x, pj + y) : 0.f;
    float T[3][3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      T[x][0] = M[x][0] * Ej.p + M[x][1] * Ej.q;
      T[x][1] = -M[x][0] * Ej.q + M[x][1] * Ej.p;
      T[x][2] = M[x][0] * Ej.u + M[x][1] * Ej.v + M[x][2];
    }
#pragma unroll
    for (int y = 0; y < 3; ++y) {
      M[0][y] = Ei.p * T[0][y] + Ei.q * T[1][y];
      M[1][y] = -Ei.q * T[0][y] + Ei.p * T[1][y];
      M[2][y] = Ei.u * T[0][y] + Ei.v * T[1][y] + T[2][y];
    }
#pragma unroll
    for (int x = 0; x < 3; ++x)
#pragma unroll
      for (int y = 0; y < 3; ++y)
        if (x < di && y < dj && (bi != bj || y <= x)) Hs[tri(pi + x, pj + y)] = M[x][y];
  }
  for (int b = lane; b < nbk; b += TEAM) {
    const int pb = bpos(b), db = b <= npn ? 3 : 2;
    const Etype E = etype(b);
    float t0[3], t1[3], t2[3] = {0, 0, 0};
#pragma unroll
    for (int y = 0; y < 3; ++y) { t0[y] = Q[3 * pb + y]; t1[y] = Q[3 * (pb + 1) + y]; if (db == 3) t2[y] = Q[3 * (pb + 2) + y]; }
    const float g0 = gam[pb], g1 = gam[pb + 1], g2 = db == 3 ? gam[pb + 2] : 0.f;
#pragma unroll
    for (int y = 0; y < 3; ++y) {
      Q[3 * pb + y] = E.p * t0[y] + E.q * t1[y];
      Q[3 * (pb + 1) + y] = -E.q * t0[y] + E.p * t1[y];
      if (db == 3) Q[3 * (pb + 2) + y] = E.u * t0[y] + E.v * t1[y] + t2[y];
    }
    gam[pb] = E.p * g0 + E.q * g1;
    gam[pb + 1] = -E.q * g0 + E.p * g1;
    if (db == 3) gam[pb + 2] = E.u * g0 + E.v * g1 + g2;
  }
  tm.sync();
  // --- I. H_ww, gamma_w (every lane redundantly), K = G[:,w] + T (into Q), KW = K H_ww^{-1} (into X)
  float Hw[3][3], gw[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) {
    gw[x] = gam[3 + x] + gx[x];
#pragma unroll
    for (int y = 0; y < 3; ++y) Hw[x][y] = sym_get(Hs, 3 + x, 3 + y) + Q[3 * (3 + x) + y] + Q[3 * (3 + y) + x] + Y[3 * x + y];
  }
  float Wi[3][3];
  {
    const float c00 = Hw[1][1] * Hw[2][2] - Hw[1][2] * Hw[2][1];
    const float c01 = Hw[1][2] * Hw[2][0] - Hw[1][0] * Hw[2][2];
    const float c02 = Hw[1][0] * Hw[2][1] - Hw[1][1] * Hw[2][0];
    const float det = Hw[0][0] * c00 + Hw[0][1] * c01 + Hw[0][2] * c02;
    const float id = 1.0f / det;
    Wi[0][0] = c00 * id; Wi[1][0] = c01 * id; Wi[2][0] = c02 * id;
    Wi[0][1] = (Hw[0][2] * Hw[2][1] - Hw[0][1] * Hw[2][2]) * id;
    Wi[1][1] = (Hw[0][0] * Hw[2][2] - Hw[0][2] * Hw[2][0]) * id;
    Wi[2][1] = (Hw[0][1] * Hw[2][0] - Hw[0][0] * Hw[2][1]) * id;
    Wi[0][2] = (Hw[0][1] * Hw[1][2] - Hw[0][2] * Hw[1][1]) * id;
    Wi[1][2] = (Hw[0][2] * Hw[1][0] - Hw[0][0] * Hw[1][2]) * id;
    Wi[2][2] = (Hw[0][0] * Hw[1][1] - Hw[0][1] * Hw[1][0]) * id;
  }
  tm.sync();
  for (int r = lane; r < s; r += TEAM) {
    if (r >= 3 && r < 6) continue;
    float K[3];
#pragma unroll
    for (int y = 0; y < 3; ++y) K[y] = Q[3 * r + y] + sym_get(Hs, r, 3 + y);
#pragma unroll
    for (int y = 0; y < 3; ++y) {
      Q[3 * r + y] = K[y];
      X[3 * r + y] = K[0] * Wi[0][y] + K[1] * Wi[1][y] + K[2] * Wi[2][y];
    }
  }
  tm.sync();
  // --- 6. re-anchor the state (A.5 step 6); slot k keeps its ring position, slot 1 becomes the frame
  {
    const float nax = w.st[0] + ddx, nay = w.st[1] + ddy, nat = wrapf(a_th + th1);
    for (int k = 2 + lane; k < c; k += TEAM) {
      float* e = w.st + st_pose(k);
      const float ex = e[0] - x1, ey = e[1] - y1;
      e[0] = c1 * ex + s1 * ey; e[1] = -s1 * ex + c1 * ey; e[2] = wrapf(e[2] - th1);
    }
    tm.sync();
    if (lane == 0) { w.st[0] = nax; w.st[1] = nay; w.st[2] = nat; }
    if (lane < 3) w.st[st_pose(1) + lane] = 0.f;
    tm.sync();
  }
  // --- J. write (Lambda', g', vbar') on the support without w, packed lower, canonical order
  {
    float* lam = rec + ly.o_lam;
    // flat over the packed triangle of the new prior (support without w): coalesced stores, every lane busy
    const int sr = s - 3, nout = sr * (sr + 1) >> 1;
    int tp = tri_row(lane), tq = lane - (tp * (tp + 1) >> 1);
    for (int t = lane; t < nout; t += TEAM) {
      const int r = tp < 3 ? tp : tp + 3, q = tq < 3 ? tq : tq + 3;
      lam[t] = Hs[tri(r, q)] - (X[3 * r] * Q[3 * q] + X[3 * r + 1] * Q[3 * q + 1] + X[3 * r + 2] * Q[3 * q + 2]);
      tri_advance(tp, tq, TEAM);
    }
    for (int r = lane; r < s; r += TEAM) {
      if (r >= 3 && r < 6) continue;
      const int R = r < 3 ? r : r - 3;
      rec[ly.o_g + R] = gam[r] - (X[3 * r] * gw[0] + X[3 * r + 1] * gw[1] + X[3 * r + 2] * gw[2]);
      rec[ly.o_vbar + R] = w.st[nidx[r] & 0xffff];
    }
  }
  // --- K. bookkeeping: loop closures to the old slot 0 now live in the prior; new support masks
  for (int k = 1 + lane; k < c; k += TEAM)
    if (w.lct[k] == 0) reci[ly.o_lct + ring_of(k, head, W)] = -1;
  mk.um &= ~1ull;       // the unary factor of the old slot 0 now lives in the prior
  mk.ps = nps & ~2ull;  // still indexed by the OLD slots; converted with the old head
  mk.ls = nls;
  if (lane == 0) {
    const uint64_t pm = slot_to_ring(mk.ps, head, W);
    recu[ly.o_pm] = (uint32_t)pm; recu[ly.o_pm + 1] = (uint32_t)(pm >> 32);
    recu[ly.o_lm] = (uint32_t)nls; recu[ly.o_lm + 1] = (uint32_t)(nls >> 32);
  }
  tm.sync();
  return 0;
}

}  // namespace slamk
