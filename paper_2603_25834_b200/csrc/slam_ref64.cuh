// fp64 path of the fixed-lag smoother: one CTA per environment, plain dense (packed lower-triangular)
// storage, straightforward loops.  Two uses:
//   1. FALLBACK for ill-conditioned windows.  The fp32 step kernel (slam_kernels.cuh) watches the
//      cancellation in the anchor's pivots, H_aa / L_aa^2 (a robot that dead-reckoned for a while and
//      re-observes a landmark: information on the anchor spans 1e0 .. 1e6, beyond fp32 -- DESIGN.md
//      section 4).  Such an environment is NOT committed by the fp32 kernel; it is appended to a list and
//      this kernel redoes the whole call for it in fp64, keeps its state and prior in an fp64 shadow
//      record, and hands it back to the fp32 kernel once the ratio has fallen again (hysteresis).
//   2. DEVICE REFERENCE: with SLAM_FORCE_FP64 every environment runs here, an independent second
//      implementation of the same mathematics (different storage, different factorisation, fp64) that the
//      tests compare the fp32 kernel with at full batch size.
// It computes exactly what DESIGN.md section 2 states (eqs. (5)-(6); readings R1-R27)
// on the same record layout (slam_layout.h): integers, masks and measurements live in the fp32 record,
// the real-valued state (a, e, g) and the prior (vbar, g, Lambda) in the record selected by `o_mode`.
// Elimination order: [passive landmarks | poses 1..W-1 except the newest | observed landmarks | newest | a].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "slam_kernels.cuh"

namespace slamr {
using slamk::Layout;
using slamk::Params;
using slamk::StepIO;
using slamk::lowmask;
using slamk::ring_of;
using slamk::ring_to_slot;
using slamk::slot_to_ring;

typedef double real;
constexpr int NT = 128;  // threads per environment (one CTA)

#ifdef SLAM_REF_PROFILE   // developer build: cycles per phase into stats[8 + slot] (read with slam_get_stats)
__device__ unsigned long long* g_ref_prof;
#define REF_TICK(slot) { __syncthreads(); if (threadIdx.x == 0) { const long long tk1 = clock64(); atomicAdd(g_ref_prof + 8 + (slot), (unsigned long long)(tk1 - ref_tk0)); ref_tk0 = clock64(); } }
#define REF_TICK_DECL long long ref_tk0 = clock64();
#else
#define REF_TICK(slot)
#define REF_TICK_DECL
#endif

struct RefArgs {
  float* state32;
  double* state64;
  int head_g, c, flags, iters;
  int* list;          // environments to process
  int* cnt;           // [0] entries in list, [1] cursor, [2] CTAs finished, [3] unused
  unsigned long long* stats;
  double* hglob;      // packed H per CTA when it does not fit shared memory (else nullptr)
  double ratio_lo;    // back to fp32 below this anchor pivot ratio
  int force;          // 1: every environment stays in fp64 (device reference)
  int min_vis;        // landmarks the newest pose must see for the hand-over back to fp32
  int box_vis;        // ... and to count as well localised (twice the thresholds; 0: never)
  int* keys;          // cost keys of the step kernel's order (see the end of the kernel), or nullptr
};

// shared-memory views of one environment
struct Sm {
  real* v;      // [n] state, natural index: a 0..2, e_k 3k.., g_l 3W+2l..
  real* b;      // [n] rhs / y / delta, elimination order
  real* d;      // [n] prior displacement on the support; scratch
  real* cs;     // [2W] cos, sin of each slot's heading (anchor frame)
  real* part;   // [max(W,L)][9] partial sums of the anchor block
  real* X;      // [3n] marginalisation: X rows
  real* Q;      // [3n] marginalisation: H_s X
  int* pos;     // [n] state index -> elimination position
  int* first;   // [n] first non-zero column of each row
  int* sidx;    // [n] support scalar -> state index
  int* omap;    // [n] old support scalar -> new support scalar
  int* lct;     // [W] loop-closure target slot or -1
  uint32_t* rbm;  // [W][nw] visibility masks by slot
  real* H;      // packed lower triangle (shared or global)
};

__host__ __device__ inline size_t ref_smem_doubles(const Layout& ly) {  // everything but H
  const int n = ly.n, m = ly.W > ly.L ? ly.W : ly.L;
  (void)m;   // (part and cs alias X, Q: 9 m + 2 W <= 6 n always)
  return (size_t)2 * n + ((n + 1) & ~1) + 6 * n + 2;
}
__host__ __device__ inline size_t ref_smem_ints(const Layout& ly) { return (size_t)4 * ly.n + ly.W + ly.W * (ly.nw ? ly.nw : 1) + 8; }
__host__ __device__ inline size_t ref_tri(const Layout& ly) { return (size_t)ly.n * (ly.n + 1) / 2; }

__device__ __forceinline__ real wrapr(real x) { return x - 6.283185307179586476925 * rint(x * 0.159154943091895335769); }
__device__ __forceinline__ int tri(int p, int q) { return (p * (p + 1) >> 1) + q; }
__device__ __forceinline__ real& Hat(real* H, int p, int q) { return p >= q ? H[tri(p, q)] : H[tri(q, p)]; }
__device__ __forceinline__ int vpose(int k) { return 3 * k; }                        // k >= 1; the anchor a is index 0
__device__ __forceinline__ int vlm(const Layout& ly, int l) { return 3 * ly.W + 2 * l; }
__device__ __forceinline__ bool is_angle(const Layout& ly, int i) { return i < 3 * ly.W && (i % 3) == 2; }
__device__ __forceinline__ int nth_bit(uint64_t m, int k) {
  for (int i = 0; i < k; ++i) m &= m - 1;
  return __ffsll((long long)m) - 1;
}

struct Ctx {  // CTA-uniform
  int env, k0, head, c, mode, s, knew;
  uint64_t ps, ls, act, um, obs;
  float* r32;
  double* r64;
};
__device__ __forceinline__ real ldr(const Ctx& e, int off) { return e.mode ? e.r64[off] : (real)e.r32[off]; }

// H(rows at pr.., cols at pc..) += M (dr x dc); `diag`: same variable, lower triangle only
template <int DR, int DC>
__device__ __forceinline__ void add_block(real* H, int pr, int pc, const real (&M)[DR][DC], bool diag) {
#pragma unroll
  for (int x = 0; x < DR; ++x)
#pragma unroll
    for (int y = 0; y < DC; ++y)
      if (!diag || y <= x) Hat(H, pr + x, pc + y) += M[x][y];
}

// between factor i -> j in the anchor frame; i_frame: pose i is the frame itself
struct Btw { real r[3], Ji[3][3], Jj[3][3]; };
__device__ __forceinline__ Btw between(const real* pi, real ci, real si, const real* pj, const float* z, bool i_frame) {
  Btw f;
  const real px = i_frame ? 0.0 : pi[0], py = i_frame ? 0.0 : pi[1], pt = i_frame ? 0.0 : pi[2];
  const real dx = pj[0] - px, dy = pj[1] - py;
  const real hx = ci * dx + si * dy, hy = -si * dx + ci * dy;
  f.r[0] = hx - (real)z[0]; f.r[1] = hy - (real)z[1]; f.r[2] = wrapr(pj[2] - pt - (real)z[2]);
  f.Jj[0][0] = ci; f.Jj[0][1] = si; f.Jj[0][2] = 0; f.Jj[1][0] = -si; f.Jj[1][1] = ci; f.Jj[1][2] = 0;
  f.Jj[2][0] = 0; f.Jj[2][1] = 0; f.Jj[2][2] = 1;
  f.Ji[0][0] = -ci; f.Ji[0][1] = -si; f.Ji[0][2] = hy; f.Ji[1][0] = si; f.Ji[1][1] = -ci; f.Ji[1][2] = -hx;
  f.Ji[2][0] = 0; f.Ji[2][1] = 0; f.Ji[2][2] = -1;
  return f;
}
// A' diag(om) B for 3-row Jacobians
template <int DA, int DB>
__device__ __forceinline__ void jtj(const real (&A)[3][DA], const real* om, const real (&B)[3][DB], real (&out)[DA][DB]) {
#pragma unroll
  for (int x = 0; x < DA; ++x)
#pragma unroll
    for (int y = 0; y < DB; ++y) out[x][y] = A[0][x] * om[0] * B[0][y] + A[1][x] * om[1] * B[1][y] + A[2][x] * om[2] * B[2][y];
}
template <int DA>
__device__ __forceinline__ void jtr(const real (&A)[3][DA], const real* om, const real* r, real (&out)[DA]) {
#pragma unroll
  for (int x = 0; x < DA; ++x) out[x] = A[0][x] * om[0] * r[0] + A[1][x] * om[1] * r[1] + A[2][x] * om[2] * r[2];
}

// range-bearing factor from slot k to landmark g (global), x = a (+) e_k (chain rule through x)
struct Rb { real r[2], Ja[2][3], Je[2][3], Jg[2][2]; };
__device__ __forceinline__ Rb rangebearing(const real* a, real ca, real sa, const real* e, bool k_frame, const real* g, real zr, real zb) {
  Rb f;
  const real ex = k_frame ? 0.0 : e[0], ey = k_frame ? 0.0 : e[1], et = k_frame ? 0.0 : e[2];
  const real ddx = ca * ex - sa * ey, ddy = sa * ex + ca * ey;      // d = Rot(a_th) t_k
  const real xx = a[0] + ddx, xy = a[1] + ddy, xt = a[2] + et;
  const real dx = g[0] - xx, dy = g[1] - xy;
  // one reciprocal square root instead of a square root and four divisions (fp64 division and sqrt are long
  // software sequences: the factor evaluation is the latency chain of the assembly)
  const real q = dx * dx + dy * dy, irho = rsqrt(q), rho = q * irho, iq = irho * irho;
  f.r[0] = rho - zr;
  f.r[1] = wrapr(atan2(dy, dx) - xt - zb);
  const real ux = dx * irho, uy = dy * irho, vx = dy * iq, vy = dx * iq;
  const real Jx[2][3] = {{-ux, -uy, 0.0}, {vx, -vy, -1.0}};
  f.Jg[0][0] = ux; f.Jg[0][1] = uy; f.Jg[1][0] = -vx; f.Jg[1][1] = vy;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    f.Ja[i][0] = Jx[i][0]; f.Ja[i][1] = Jx[i][1]; f.Ja[i][2] = -Jx[i][0] * ddy + Jx[i][1] * ddx + Jx[i][2];
    f.Je[i][0] = Jx[i][0] * ca + Jx[i][1] * sa; f.Je[i][1] = -Jx[i][0] * sa + Jx[i][1] * ca; f.Je[i][2] = Jx[i][2];
  }
  return f;
}

__device__ inline Sm carve(const Layout& ly, double* base, double* hglob) {
  Sm s;
  const int n = ly.n, m = ly.W > ly.L ? ly.W : ly.L;
  double* p = base;
  s.v = p; p += n; s.b = p; p += n; s.d = p; p += (n + 1) & ~1;   // (X 16-byte aligned: 128-bit loads in ref_cholesky)
  s.X = p; p += 3 * n; s.Q = p; p += 3 * n; p += 2;
  // only ref_assemble needs the partial sums and the cos / sin table, and nothing else lives in X, Q while it runs
  // (ref_cholesky's compact columns and the marginalisation come later): they share that storage, which is what
  // lets FOUR environments fit an SM at config 3
  s.part = s.X; s.cs = s.X + ((9 * m + 1) & ~1);
  int* q = reinterpret_cast<int*>(p);
  s.pos = q; q += n; s.first = q; q += n; s.sidx = q; q += n; s.omap = q; q += n; s.lct = q; q += ly.W;
  s.rbm = reinterpret_cast<uint32_t*>(q); q += ly.W * (ly.nw ? ly.nw : 1); q += 8;
  q = reinterpret_cast<int*>((reinterpret_cast<uintptr_t>(q) + 15) & ~(uintptr_t)15);
  s.H = hglob ? hglob : reinterpret_cast<double*>(q);
  return s;
}

__device__ __forceinline__ uint64_t vis_of(const Layout& ly, const Sm& s, int k) {
  uint64_t m = (uint64_t)s.rbm[k * ly.nw];
  if (ly.nw > 1) m |= (uint64_t)s.rbm[k * ly.nw + 1] << 32;
  return m;
}

// ------------------------------------------------------------------ load / push
__device__ void ref_load(const Layout& ly, Ctx& e, const Sm& s, int tid) {
  const int W = ly.W, L = ly.L;
  const int* ri = reinterpret_cast<const int*>(e.r32);
  const uint32_t* ru = reinterpret_cast<const uint32_t*>(e.r32);
  for (int i = tid; i < 3 * W; i += NT) {
    const int k = i / 3, j = i - 3 * k;
    real val;
    if (k == 0) val = ldr(e, ly.o_a + j);
    else val = k < e.c ? ldr(e, ly.o_e + 3 * ring_of(k, e.head, W) + j) : 0.0;
    s.v[i] = val;
  }
  for (int i = tid; i < 2 * L; i += NT) s.v[3 * W + i] = ldr(e, ly.o_m + i);
  for (int k = tid; k < W; k += NT) {
    const int r = ring_of(k, e.head, W);
    const int t = k < e.c ? ri[ly.o_lct + r] : -1;
    int ts = -1;
    if (t >= 0) { ts = t - e.head; if (ts < 0) ts += W; }
    s.lct[k] = ts;
    for (int q = 0; q < ly.nw; ++q) s.rbm[k * ly.nw + q] = k < e.c ? ru[ly.o_rbm + r * ly.nw + q] : 0u;
  }
  const uint64_t pm = (uint64_t)ru[ly.o_pm] | ((uint64_t)ru[ly.o_pm + 1] << 32);
  e.ps = ring_to_slot(pm, e.head, W);
  e.ls = (uint64_t)ru[ly.o_lm] | ((uint64_t)ru[ly.o_lm + 1] << 32);
  e.act = (uint64_t)ru[ly.o_act] | ((uint64_t)ru[ly.o_act + 1] << 32);
  e.um = ring_to_slot((uint64_t)ru[ly.o_um] | ((uint64_t)ru[ly.o_um + 1] << 32), e.head, W) & lowmask(e.c);
  __syncthreads();
}

// range-bearing bookkeeping of the pose in `slot` (pose p in the anchor frame): measurements into the record,
// newly seen landmarks initialised by inverse projection from the pose's current guess (reading R6)
__device__ void ref_record_rb(const Layout& ly, Ctx& e, const Sm& s, int tid, int slot, real px, real py, real pth, const StepIO& io) {
  const int L = ly.L, N = ly.N, r = ring_of(slot, e.head, ly.W);
  uint32_t* ru = reinterpret_cast<uint32_t*>(e.r32);
  uint64_t vis = (uint64_t)io.rb_mask[e.env];
  if (ly.nw > 1) vis |= (uint64_t)io.rb_mask[(size_t)N + e.env] << 32;
  vis &= lowmask(L);
  const real sa = sin(s.v[2]), ca = cos(s.v[2]);
  const real gx = s.v[0] + ca * px - sa * py, gy = s.v[1] + sa * px + ca * py, gt = s.v[2] + pth;
  __syncthreads();
  for (int l = tid; l < L; l += NT) {
    const float zr = io.rb_meas[(size_t)l * N + e.env], zb = io.rb_meas[(size_t)(L + l) * N + e.env];
    e.r32[ly.o_zrb + (r * 2 + 0) * L + l] = zr;
    e.r32[ly.o_zrb + (r * 2 + 1) * L + l] = zb;
    if (((vis >> l) & 1ull) && !((e.act >> l) & 1ull)) {
      s.v[vlm(ly, l)] = gx + (real)zr * cos(gt + (real)zb);
      s.v[vlm(ly, l) + 1] = gy + (real)zr * sin(gt + (real)zb);
    }
  }
  if (tid < ly.nw) {
    const uint32_t word = (uint32_t)(vis >> (32 * tid));
    s.rbm[slot * ly.nw + tid] = word;
    ru[ly.o_rbm + r * ly.nw + tid] = word;
  }
  e.act |= vis;
  __syncthreads();
}

__device__ void ref_push(const Layout& ly, Ctx& e, const Sm& s, int tid, const StepIO& io) {
  const int W = ly.W, N = ly.N, c = e.c, r = ring_of(c, e.head, W);
  int* ri = reinterpret_cast<int*>(e.r32);
  const float zx = io.odom[e.env], zy = io.odom[(size_t)N + e.env], zt = io.odom[2 * (size_t)N + e.env];
  const real pxo = c > 1 ? s.v[vpose(c - 1)] : 0.0, pyo = c > 1 ? s.v[vpose(c - 1) + 1] : 0.0, pto = c > 1 ? s.v[vpose(c - 1) + 2] : 0.0;
  const real sn = sin(pto), cn = cos(pto);
  const real nx = pxo + cn * (real)zx - sn * (real)zy, ny = pyo + sn * (real)zx + cn * (real)zy, nt = wrapr(pto + (real)zt);
  const int back = io.lc_back ? io.lc_back[e.env] : 0;
  const int tgt = (back >= 1 && back <= c) ? c - back : -1;  // R11
  __syncthreads();
  if (tid == 0) {
    s.v[vpose(c)] = nx; s.v[vpose(c) + 1] = ny; s.v[vpose(c) + 2] = nt;
    s.lct[c] = tgt;
    ri[ly.o_lct + r] = tgt < 0 ? -1 : ring_of(tgt, e.head, W);
  }
  if (tid < 3) {
    e.r32[ly.o_zodo + 3 * r + tid] = tid == 0 ? zx : (tid == 1 ? zy : zt);
    e.r32[ly.o_zlc + 3 * r + tid] = io.lc_meas ? io.lc_meas[(size_t)tid * N + e.env] : 0.0f;
  }
  e.um &= ~(1ull << c);
  if (io.un_pose && (io.un_valid == nullptr || io.un_valid[e.env] != 0)) {
    if (tid < 3) e.r32[ly.o_zun + 3 * r + tid] = io.un_pose[(size_t)tid * N + e.env];
    if (tid < 6) e.r32[ly.o_omun + 6 * r + tid] = io.un_info[(size_t)tid * N + e.env];
    e.um |= 1ull << c;
  }
  __syncthreads();
  if (ly.L > 0) ref_record_rb(ly, e, s, tid, c, nx, ny, nt, io);
  e.c = c + 1;
}

// ------------------------------------------------------------------ order and prior support
__device__ void ref_order(const Layout& ly, Ctx& e, const Sm& s, int tid) {
  const int W = ly.W, L = ly.L, n = ly.n;
  uint64_t obs = 0ull;
  for (int k = 0; k < e.c; ++k) obs |= vis_of(ly, s, k);
  e.obs = obs & lowmask(L);
  const int npas = L - __popcll(e.obs);
  e.knew = e.c >= 2 ? e.c - 1 : W - 1;
  const int oC = 2 * npas, oL = oC + 3 * (W - 2), oN = n - 6, oA = n - 3;
  for (int i = tid; i < n; i += NT) {
    int p;
    if (i < 3) p = oA + i;
    else if (i < 3 * W) {
      const int k = i / 3, j = i - 3 * k;
      p = k == e.knew ? oN + j : oC + 3 * (k < e.knew ? k - 1 : k - 2) + j;
    } else {
      const int l = (i - 3 * W) >> 1, j = (i - 3 * W) & 1;
      const uint64_t below = lowmask(l);
      p = ((e.obs >> l) & 1ull) ? oL + 2 * __popcll(e.obs & below) + j : 2 * __popcll(~e.obs & below) + j;
    }
    s.pos[i] = p;
  }
  // support table, canonical order [a | support pose slots ascending | support landmarks ascending]
  const int npo = __popcll(e.ps), nlo = __popcll(e.ls);
  e.s = 3 + 3 * npo + 2 * nlo;
  for (int p = tid; p < e.s; p += NT) {
    int idx;
    if (p < 3) idx = p;
    else if (p < 3 + 3 * npo) { const int bk = (p - 3) / 3; idx = vpose(nth_bit(e.ps, bk)) + (p - 3 - 3 * bk); }
    else { const int q = p - 3 - 3 * npo; idx = vlm(ly, nth_bit(e.ls, q >> 1)) + (q & 1); }
    s.sidx[p] = idx;
  }
  __syncthreads();
}

// ------------------------------------------------------------------ assemble H, b at the current state
__device__ void ref_assemble(const Layout& ly, const Params& pr, const Ctx& e, const Sm& s, int tid) {
  const int W = ly.W, L = ly.L, n = ly.n, c = e.c;
  REF_TICK_DECL
  real* H = s.H;
  const int ntri = n * (n + 1) / 2;
  for (int t = tid; t < ntri; t += NT) H[t] = 0.0;
  for (int i = tid; i < n; i += NT) s.b[i] = 0.0;
  for (int k = tid; k < W; k += NT) {
    real sn = 0.0, cn = 1.0;
    if (k > 0 && k < c) { sn = sin(s.v[vpose(k) + 2]); cn = cos(s.v[vpose(k) + 2]); }
    s.cs[2 * k] = cn; s.cs[2 * k + 1] = sn;
  }
  for (int p = tid; p < e.s; p += NT) {
    real d = s.v[s.sidx[p]] - ldr(e, ly.o_vbar + p);
    if (is_angle(ly, s.sidx[p])) d = wrapr(d);
    s.d[p] = d;
  }
  __syncthreads();
  REF_TICK(0)
  // prior: H = Lambda on the support; b = -(Lambda d + g) read back from shared memory (no second pass over HBM)
  {
    const int st = e.s * (e.s + 1) / 2;
    if (tid < st) {  // (row, column) of this thread's first entry by one square root, then advanced NT entries at a time
      int p = (int)((sqrtf(8.0f * (float)tid + 1.0f) - 1.0f) * 0.5f);
      while ((p + 1) * (p + 2) / 2 <= tid) ++p;
      while (p * (p + 1) / 2 > tid) --p;
      int q = tid - p * (p + 1) / 2;
      for (int t = tid;;) {
        Hat(H, s.pos[s.sidx[p]], s.pos[s.sidx[q]]) = ldr(e, ly.o_lam + t);
        t += NT;
        if (t >= st) break;
        q += NT;
        while (q > p) { q -= p + 1; ++p; }
      }
    }
    __syncthreads();
    for (int p = tid; p < e.s; p += NT) {
      const int pp = s.pos[s.sidx[p]];
      real acc = ldr(e, ly.o_g + p);
      for (int q = 0; q < e.s; ++q) acc += Hat(H, pp, s.pos[s.sidx[q]]) * s.d[q];
      s.b[pp] = -acc;
    }
  }
  // identity rows: unused pose slots, inactive landmarks
  for (int i = 3 + tid; i < n; i += NT) {
    const bool unused = i < 3 * W ? (i / 3) >= c : !((e.act >> ((i - 3 * W) >> 1)) & 1ull);
    if (unused) H[tri(s.pos[i], s.pos[i])] = 1.0;
  }
  __syncthreads();
  REF_TICK(1)
  // odometry k-1 -> k: j side, then i side
  const real om_odo[3] = {pr.om_odo[0], pr.om_odo[1], pr.om_odo[2]}, om_lc[3] = {pr.om_lc[0], pr.om_lc[1], pr.om_lc[2]};
  for (int pass = 0; pass < 2; ++pass) {
    for (int k = 1 + tid; k < c; k += NT) {
      const Btw f = between(s.v + vpose(k - 1), s.cs[2 * (k - 1)], s.cs[2 * (k - 1) + 1], s.v + vpose(k),
                            e.r32 + ly.o_zodo + 3 * ring_of(k, e.head, W), k == 1);
      const int pj = s.pos[vpose(k)];
      if (pass == 0) {
        real M[3][3], g[3];
        jtj(f.Jj, om_odo, f.Jj, M); add_block(H, pj, pj, M, true);
        jtr(f.Jj, om_odo, f.r, g);
        for (int x = 0; x < 3; ++x) s.b[pj + x] -= g[x];
        if (k >= 2) { jtj(f.Jj, om_odo, f.Ji, M); add_block(H, pj, s.pos[vpose(k - 1)], M, false); }
      } else if (k >= 2) {
        const int pi = s.pos[vpose(k - 1)];
        real M[3][3], g[3];
        jtj(f.Ji, om_odo, f.Ji, M); add_block(H, pi, pi, M, true);
        jtr(f.Ji, om_odo, f.r, g);
        for (int x = 0; x < 3; ++x) s.b[pi + x] -= g[x];
      }
    }
    __syncthreads();
  }
  REF_TICK(2)
  // loop closures t -> k: j side (one per k), i side (thread per target, serial over its sources)
  for (int k = 1 + tid; k < c; k += NT) {
    const int t = s.lct[k];
    if (t < 0) continue;
    const Btw f = between(s.v + vpose(t), s.cs[2 * t], s.cs[2 * t + 1], s.v + vpose(k), e.r32 + ly.o_zlc + 3 * ring_of(k, e.head, W), t == 0);
    const int pj = s.pos[vpose(k)];
    real M[3][3], g[3];
    jtj(f.Jj, om_lc, f.Jj, M); add_block(H, pj, pj, M, true);
    jtr(f.Jj, om_lc, f.r, g);
    for (int x = 0; x < 3; ++x) s.b[pj + x] -= g[x];
    if (t >= 1) { jtj(f.Jj, om_lc, f.Ji, M); add_block(H, pj, s.pos[vpose(t)], M, false); }
  }
  __syncthreads();
  for (int t = 1 + tid; t < c - 1; t += NT) {
    const int pi = s.pos[vpose(t)];
    for (int k = t + 1; k < c; ++k) {
      if (s.lct[k] != t) continue;
      const Btw f = between(s.v + vpose(t), s.cs[2 * t], s.cs[2 * t + 1], s.v + vpose(k), e.r32 + ly.o_zlc + 3 * ring_of(k, e.head, W), false);
      real M[3][3], g[3];
      jtj(f.Ji, om_lc, f.Ji, M); add_block(H, pi, pi, M, true);
      jtr(f.Ji, om_lc, f.r, g);
      for (int x = 0; x < 3; ++x) s.b[pi + x] -= g[x];
    }
  }
  __syncthreads();
  const int oA = n - 3;
  const real sa = sin(s.v[2]), ca = cos(s.v[2]);
  REF_TICK(3)
  // unary absolute-pose factors: r = (a (+) e_k) - z, full 3x3 information
  if (e.um) {
    for (int k = tid; k < W; k += NT) {
      real* P = s.part + 9 * k;
      for (int x = 0; x < 9; ++x) P[x] = 0.0;
      if (k >= c || !((e.um >> k) & 1ull)) continue;
      const int r = ring_of(k, e.head, W);
      const real ex = k ? s.v[vpose(k)] : 0.0, ey = k ? s.v[vpose(k) + 1] : 0.0, et = k ? s.v[vpose(k) + 2] : 0.0;
      const real dx = ca * ex - sa * ey, dy = sa * ex + ca * ey;
      const real res[3] = {s.v[0] + dx - (real)e.r32[ly.o_zun + 3 * r], s.v[1] + dy - (real)e.r32[ly.o_zun + 3 * r + 1],
                           wrapr(s.v[2] + et - (real)e.r32[ly.o_zun + 3 * r + 2])};
      const float* o6 = e.r32 + ly.o_omun + 6 * r;
      const real O[3][3] = {{o6[0], o6[1], o6[3]}, {o6[1], o6[2], o6[4]}, {o6[3], o6[4], o6[5]}};
      const real Ja[3][3] = {{1.0, 0.0, -dy}, {0.0, 1.0, dx}, {0.0, 0.0, 1.0}};
      const real Je[3][3] = {{ca, -sa, 0.0}, {sa, ca, 0.0}, {0.0, 0.0, 1.0}};
      real Or[3], OJa[3][3], OJe[3][3];
      for (int i = 0; i < 3; ++i) {
        Or[i] = O[i][0] * res[0] + O[i][1] * res[1] + O[i][2] * res[2];
        for (int j = 0; j < 3; ++j) {
          OJa[i][j] = O[i][0] * Ja[0][j] + O[i][1] * Ja[1][j] + O[i][2] * Ja[2][j];
          OJe[i][j] = O[i][0] * Je[0][j] + O[i][1] * Je[1][j] + O[i][2] * Je[2][j];
        }
      }
      int t = 0;
      for (int x = 0; x < 3; ++x) {
        for (int y = 0; y <= x; ++y) P[t++] = Ja[0][x] * OJa[0][y] + Ja[1][x] * OJa[1][y] + Ja[2][x] * OJa[2][y];
        P[6 + x] = Ja[0][x] * Or[0] + Ja[1][x] * Or[1] + Ja[2][x] * Or[2];
      }
      if (k >= 1) {
        const int pe = s.pos[vpose(k)];
        for (int x = 0; x < 3; ++x) {
          for (int y = 0; y <= x; ++y) Hat(H, pe + x, pe + y) += Je[0][x] * OJe[0][y] + Je[1][x] * OJe[1][y] + Je[2][x] * OJe[2][y];
          for (int y = 0; y < 3; ++y) Hat(H, oA + x, pe + y) += Ja[0][x] * OJe[0][y] + Ja[1][x] * OJe[1][y] + Ja[2][x] * OJe[2][y];
          s.b[pe + x] -= Je[0][x] * Or[0] + Je[1][x] * Or[1] + Je[2][x] * Or[2];
        }
      }
    }
    __syncthreads();
    if (tid < 9) {
      real acc = 0.0;
      for (int k = 0; k < c; ++k) acc += s.part[9 * k + tid];
      if (tid < 6) { const int x = tid < 1 ? 0 : (tid < 3 ? 1 : 2), y = tid - (x * (x + 1) >> 1); H[tri(oA + x, oA + y)] += acc; }
      else s.b[oA + tid - 6] -= acc;
    }
    __syncthreads();
  }
  // range-bearing factors.  Pass A: thread per observing pose (pose block, pose x landmark, anchor x pose);
  // pass B: thread per landmark (landmark block, anchor x landmark, partial sums of the anchor block)
  if (L > 0 && e.obs) {
    const real om_rb[3] = {pr.om_rb[0], pr.om_rb[1], 0.0};
    // four adjacent lanes share one pose (pass A) / one landmark (pass B): each takes every fourth factor, the
    // partial sums are combined by shuffles in a fixed order (deterministic)
    const int grp = tid >> 2, sub = tid & 3;
    for (int k0 = 1; k0 < c; k0 += NT / 4) {
      const int k = k0 + grp;
      uint64_t m = k < c ? vis_of(ly, s, k) : 0ull;
      const bool any = m != 0ull;
      const int r = ring_of(k < c ? k : 0, e.head, W), pe = k < c ? s.pos[vpose(k)] : 0;
      real E[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, AE[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, be[3] = {0, 0, 0};
      for (int cnt = 0; m; ++cnt) {
        const int l = __ffsll((long long)m) - 1;
        m &= m - 1;
        if ((cnt & 3) != sub) continue;
        const Rb f = rangebearing(s.v, ca, sa, s.v + vpose(k), false, s.v + vlm(ly, l), (real)e.r32[ly.o_zrb + (r * 2 + 0) * L + l],
                                  (real)e.r32[ly.o_zrb + (r * 2 + 1) * L + l]);
        real GE[2][3];
        for (int x = 0; x < 3; ++x) {
          for (int y = 0; y < 3; ++y) {
            E[x][y] += f.Je[0][x] * om_rb[0] * f.Je[0][y] + f.Je[1][x] * om_rb[1] * f.Je[1][y];
            AE[x][y] += f.Ja[0][x] * om_rb[0] * f.Je[0][y] + f.Ja[1][x] * om_rb[1] * f.Je[1][y];
          }
          be[x] += f.Je[0][x] * om_rb[0] * f.r[0] + f.Je[1][x] * om_rb[1] * f.r[1];
        }
        for (int x = 0; x < 2; ++x)
          for (int y = 0; y < 3; ++y) GE[x][y] = f.Jg[0][x] * om_rb[0] * f.Je[0][y] + f.Jg[1][x] * om_rb[1] * f.Je[1][y];
        add_block(H, s.pos[vlm(ly, l)], pe, GE, false);
      }
#pragma unroll
      for (int o = 1; o < 4; o <<= 1) {
#pragma unroll
        for (int x = 0; x < 3; ++x) {
#pragma unroll
          for (int y = 0; y < 3; ++y) {
            E[x][y] += __shfl_xor_sync(0xffffffffu, E[x][y], o);
            AE[x][y] += __shfl_xor_sync(0xffffffffu, AE[x][y], o);
          }
          be[x] += __shfl_xor_sync(0xffffffffu, be[x], o);
        }
      }
      if (any && sub == 0) {
        add_block(H, pe, pe, E, true);
        add_block(H, oA, pe, AE, false);
        for (int x = 0; x < 3; ++x) s.b[pe + x] -= be[x];
      }
    }
    __syncthreads();
    REF_TICK(4)
    for (int l0 = 0; l0 < L; l0 += NT / 4) {
      const int l = l0 + grp;
      const bool on = l < L && ((e.obs >> l) & 1ull);
      real P9[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
      real GG[2][2] = {{0, 0}, {0, 0}}, AG[3][2] = {{0, 0}, {0, 0}, {0, 0}}, bg[2] = {0, 0};
      if (on) {
        int cnt = 0;
        for (int k = 0; k < c; ++k) {
          if (!((s.rbm[k * ly.nw + (l >> 5)] >> (l & 31)) & 1u)) continue;
          if (((cnt++) & 3) != sub) continue;
          const int r = ring_of(k, e.head, W);
          const Rb f = rangebearing(s.v, ca, sa, s.v + vpose(k), k == 0, s.v + vlm(ly, l), (real)e.r32[ly.o_zrb + (r * 2 + 0) * L + l],
                                    (real)e.r32[ly.o_zrb + (r * 2 + 1) * L + l]);
          for (int x = 0; x < 2; ++x) {
            for (int y = 0; y < 2; ++y) GG[x][y] += f.Jg[0][x] * om_rb[0] * f.Jg[0][y] + f.Jg[1][x] * om_rb[1] * f.Jg[1][y];
            bg[x] += f.Jg[0][x] * om_rb[0] * f.r[0] + f.Jg[1][x] * om_rb[1] * f.r[1];
          }
          int t = 0;
          for (int x = 0; x < 3; ++x) {
            for (int y = 0; y < 2; ++y) AG[x][y] += f.Ja[0][x] * om_rb[0] * f.Jg[0][y] + f.Ja[1][x] * om_rb[1] * f.Jg[1][y];
            for (int y = 0; y <= x; ++y) P9[t++] += f.Ja[0][x] * om_rb[0] * f.Ja[0][y] + f.Ja[1][x] * om_rb[1] * f.Ja[1][y];
            P9[6 + x] += f.Ja[0][x] * om_rb[0] * f.r[0] + f.Ja[1][x] * om_rb[1] * f.r[1];
          }
        }
      }
#pragma unroll
      for (int o = 1; o < 4; o <<= 1) {
#pragma unroll
        for (int x = 0; x < 9; ++x) P9[x] += __shfl_xor_sync(0xffffffffu, P9[x], o);
#pragma unroll
        for (int x = 0; x < 2; ++x) {
#pragma unroll
          for (int y = 0; y < 2; ++y) GG[x][y] += __shfl_xor_sync(0xffffffffu, GG[x][y], o);
          bg[x] += __shfl_xor_sync(0xffffffffu, bg[x], o);
        }
#pragma unroll
        for (int x = 0; x < 3; ++x)
#pragma unroll
          for (int y = 0; y < 2; ++y) AG[x][y] += __shfl_xor_sync(0xffffffffu, AG[x][y], o);
      }
      if (l < L && sub == 0) {
        real* P = s.part + 9 * l;
        for (int x = 0; x < 9; ++x) P[x] = P9[x];
        if (on) {
          const int pg = s.pos[vlm(ly, l)];
          add_block(H, pg, pg, GG, true);
          add_block(H, oA, pg, AG, false);
          s.b[pg] -= bg[0]; s.b[pg + 1] -= bg[1];
        }
      }
    }
    __syncthreads();
    if (tid < 9) {
      real acc = 0.0;
      for (int l = 0; l < L; ++l) acc += s.part[9 * l + tid];
      if (tid < 6) { const int x = tid < 1 ? 0 : (tid < 3 ? 1 : 2), y = tid - (x * (x + 1) >> 1); H[tri(oA + x, oA + y)] += acc; }
      else s.b[oA + tid - 6] -= acc;
    }
    __syncthreads();
  }
  REF_TICK(5)
}

// ------------------------------------------------------------------ Cholesky (right-looking, blocks of 4 columns)
// Per block: the rows with entries in the block scale their four entries with the block's factorised 4x4 tile and
// are gathered in a compact list; the rank-4 update of the trailing envelope runs over 2x2 tiles of that list.
// LOOK-AHEAD: while warps 1.. update the trailing envelope, the first warp applies the update to the NEXT block's
// diagonal tile (the pairs among the first four list entries), factorises it (and the rhs entries of that block)
// in registers and publishes it in the other of two buffers -- the four dependent fp64 rsqrt of a tile (~700 cycles)
// are off the critical path, and a block costs two CTA barriers instead of three.
// On exit H holds L (diagonal = L_jj), b holds y = L^{-1} b, s.d holds 1 / L_jj.
// Returns status bits; *ratio = max over the anchor rows of H_ii / L_ii^2 (the cancellation the fp32 kernel
// cannot afford).
struct RefTile { real t[4][4], ti[4], y[4]; };

// first warp: factorise the tile of block j (nb columns), identity-padded when nb < 4 (every lane the same arithmetic)
__device__ __forceinline__ int ref_factor_tile(real* H, real* b, real* dinv, int j, int nb, int lane, RefTile* out) {
  real t[4][4], y[4], ti[4];
  int flag = 0;
#pragma unroll
  for (int x = 0; x < 4; ++x) {
#pragma unroll
    for (int c = 0; c < 4; ++c) t[x][c] = (x < nb && c <= x) ? H[tri(j + x, j + c)] : (x == c ? 1.0 : 0.0);
    y[x] = x < nb ? b[j + x] : 0.0;
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    real piv = t[c][c];
#pragma unroll
    for (int k = 0; k < c; ++k) piv -= t[c][k] * t[c][k];
    if (!(piv > 0.0)) { flag |= slamk::ENV_NOT_PD; piv = 1.0; }
    const real inv = rsqrt(piv);
    t[c][c] = piv * inv; ti[c] = inv;
#pragma unroll
    for (int x = c + 1; x < 4; ++x) {
      real v = t[x][c];
#pragma unroll
      for (int k = 0; k < c; ++k) v -= t[x][k] * t[c][k];
      t[x][c] = v * inv;
    }
    real yy = y[c];
#pragma unroll
    for (int k = 0; k < c; ++k) yy -= t[c][k] * y[k];
    y[c] = yy * inv;
  }
  __syncwarp();   // every lane has read the tile before lane 0 overwrites it
  if (lane == 0) {
#pragma unroll
    for (int x = 0; x < 4; ++x) {
#pragma unroll
      for (int c = 0; c < 4; ++c) out->t[x][c] = t[x][c];
      out->ti[x] = ti[x]; out->y[x] = y[x];
      if (x < nb) {
#pragma unroll
        for (int c = 0; c <= x; ++c) H[tri(j + x, j + c)] = t[x][c];
        b[j + x] = y[x];
        dinv[j + x] = ti[x];
      }
    }
  }
  return flag;
}

__device__ int ref_cholesky(const Layout& ly, const Sm& s, int tid, real* ratio) {
  static_assert(NT >= 64, "the look-ahead needs a second warp");
  const int n = ly.n;
  real* H = s.H;
  // L(i, j..j+3) of the active rows, component-major and compact: cmp[x * NC + position in the list] (X and Q are
  // contiguous: 6n doubles; only the marginalisation uses them as X, Q)
  real* cmp = s.X;
  const int NC = (n + 3) & ~1;
  real* dinv = s.d;   // 1 / L_jj for the back substitution (the prior displacement is dead by now)
  int* act = s.omap;  // compact list of the rows that take part in the current block
  for (int p = tid; p < n; p += NT) {  // envelope: first non-zero of each row (fill stays inside it)
    int f = 0;
    while (f < p && H[tri(p, f)] == 0.0) ++f;
    s.first[p] = f;
  }
  real ha[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) ha[x] = H[tri(n - 3 + x, n - 3 + x)];
  int flag = 0;
  __shared__ int sh_cnt[3][NT / 32];   // active rows per (chunk of NT rows, warp)
  __shared__ RefTile sh_tile[2];       // the current block's factorised tile and the next one's (look-ahead)
  __shared__ int sh_flag;
  const int lane = tid & 31, wid = tid >> 5;
  __syncthreads();
  // rows below block [j, r0) that have entries in it (first < r0): ballots for the list of the rows phase
  unsigned bal[3];
  auto ballots = [&](int r0) {
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      const int i = r0 + ch * NT + tid;
      bal[ch] = __ballot_sync(0xffffffffu, i < n && s.first[i] < r0);
      if (lane == 0) sh_cnt[ch][wid] = __popc(bal[ch]);
    }
  };
  {
    const int nb0 = n < 4 ? n : 4;
    ballots(nb0);
    if (wid == 0) flag |= ref_factor_tile(H, s.b, dinv, 0, nb0, lane, &sh_tile[0]);
  }
  __syncthreads();
  int cur = 0;
  for (int j = 0; j < n; j += 4, cur ^= 1) {
    const int nb = n - j < 4 ? n - j : 4, r0 = j + nb;
    const RefTile& T = sh_tile[cur];
    // active rows: L(i, j..j+3) by forward substitution with the tile; the rhs rides along
    int m = 0;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      int base = m;
#pragma unroll
      for (int w2 = 0; w2 < NT / 32; ++w2) { const int cw = sh_cnt[ch][w2]; if (w2 < wid) base += cw; m += cw; }
      if ((bal[ch] >> lane) & 1u) {
        const int i = r0 + ch * NT + tid;
        real* hp = H + tri(i, j);
        const real l0 = hp[0] * T.ti[0];
        real l1 = 0.0, l2 = 0.0, l3 = 0.0;
        if (nb > 1) l1 = (hp[1] - l0 * T.t[1][0]) * T.ti[1];
        if (nb > 2) l2 = (hp[2] - l0 * T.t[2][0] - l1 * T.t[2][1]) * T.ti[2];
        if (nb > 3) l3 = (hp[3] - l0 * T.t[3][0] - l1 * T.t[3][1] - l2 * T.t[3][2]) * T.ti[3];
        hp[0] = l0;
        if (nb > 1) hp[1] = l1;
        if (nb > 2) hp[2] = l2;
        if (nb > 3) hp[3] = l3;
        const int at = base + __popc(bal[ch] & ((1u << lane) - 1u));   // position in the compact list (ascending rows)
        cmp[at] = l0; cmp[NC + at] = l1; cmp[2 * NC + at] = l2; cmp[3 * NC + at] = l3;
        s.b[i] -= l0 * T.y[0] + l1 * T.y[1] + l2 * T.y[2] + l3 * T.y[3];
        act[at] = i;
      }
    }
    __syncthreads();
    // rank-4 update of the trailing envelope in 2 x 2 tiles of list positions (rows 2a, 2a+1 x columns 2b, 2b+1,
    // b <= a): the eight loads of a tile are 128-bit, the row side a broadcast and the column side contiguous over the
    // lanes (conflict-free), a quarter of the shared-memory traffic of one pair per thread (measured: a flat update
    // was bound by the LSU, 24 wavefronts per pair).
    const int m2 = (m + 1) >> 1, ntile = m2 * (m2 + 1) >> 1;
    if (wid == 0) {
      // look-ahead: the list is ascending, so the rows of the next block that are in it are among its first four
      // entries; the pairs among those four (= the 2x2 tiles 0, 1, 2) are updated here, one pair per lane, then the
      // next tile is factorised
      if (lane < 10) {
        const int pp = lane >= 6 ? 3 : (lane >= 3 ? 2 : (lane >= 1 ? 1 : 0)), qq = lane - (pp * (pp + 1) >> 1);
        if (pp < m) {
          const int i = act[pp], k = act[qq];
          H[tri(i, k)] -= cmp[pp] * cmp[qq] + cmp[NC + pp] * cmp[NC + qq] + cmp[2 * NC + pp] * cmp[2 * NC + qq] +
                          cmp[3 * NC + pp] * cmp[3 * NC + qq];
        }
      }
      __syncwarp();
      if (r0 < n) flag |= ref_factor_tile(H, s.b, dinv, r0, n - r0 < 4 ? n - r0 : 4, lane, &sh_tile[cur ^ 1]);
    } else if (ntile > 3) {
      // the other warps: tiles 3.. ; the (a, b) of this thread's first tile by one square root, then advanced
      constexpr int NU = NT - 32;
      const int t0 = 3 + tid - 32;
      if (t0 < ntile) {
        int a = (int)((sqrtf(8.0f * (float)t0 + 1.0f) - 1.0f) * 0.5f);
        if ((a + 1) * (a + 2) / 2 <= t0) ++a;
        if (a * (a + 1) / 2 > t0) --a;
        int bq = t0 - (a * (a + 1) >> 1);
        for (int p = t0;;) {
          const int ia = 2 * a, ib = 2 * bq;
          const double2 A0 = *reinterpret_cast<const double2*>(cmp + ia), A1 = *reinterpret_cast<const double2*>(cmp + NC + ia);
          const double2 A2 = *reinterpret_cast<const double2*>(cmp + 2 * NC + ia), A3 = *reinterpret_cast<const double2*>(cmp + 3 * NC + ia);
          const double2 B0 = *reinterpret_cast<const double2*>(cmp + ib), B1 = *reinterpret_cast<const double2*>(cmp + NC + ib);
          const double2 B2 = *reinterpret_cast<const double2*>(cmp + 2 * NC + ib), B3 = *reinterpret_cast<const double2*>(cmp + 3 * NC + ib);
          const bool ra1 = ia + 1 < m, cb1 = ib + 1 < m;
          const int i0 = act[ia], i1 = ra1 ? act[ia + 1] : 0, k0 = act[ib], k1 = cb1 ? act[ib + 1] : 0;
          H[tri(i0, k0)] -= A0.x * B0.x + A1.x * B1.x + A2.x * B2.x + A3.x * B3.x;
          if (ra1) H[tri(i1, k0)] -= A0.y * B0.x + A1.y * B1.x + A2.y * B2.x + A3.y * B3.x;
          if (cb1 && bq < a) H[tri(i0, k1)] -= A0.x * B0.y + A1.x * B1.y + A2.x * B2.y + A3.x * B3.y;   // (above the diagonal when b == a)
          if (ra1 && cb1) H[tri(i1, k1)] -= A0.y * B0.y + A1.y * B1.y + A2.y * B2.y + A3.y * B3.y;
          p += NU;
          if (p >= ntile) break;
          bq += NU;
          while (bq > a) { bq -= a + 1; ++a; }
        }
      }
    }
    // the list of the next block (the readers of sh_cnt of this block are past the barrier above)
    if (r0 < n) ballots(r0 + (n - r0 < 4 ? n - r0 : 4));
    __syncthreads();
  }
  real r = 0.0;
#pragma unroll
  for (int x = 0; x < 3; ++x) { const real l = H[tri(n - 3 + x, n - 3 + x)]; r = fmax(r, ha[x] / (l * l)); }
  if (tid == 0) { *ratio = fmax(*ratio, r); sh_flag = flag; }   // (thread 0 is in the warp that factorised the tiles)
  __syncthreads();
  return sh_flag;
}

// L' delta = y, in place in b: blocks of 4 rows from the bottom; the 4x4 tile solve is done by every thread
__device__ void ref_backsub(const Layout& ly, const Sm& s, int tid) {
  const int n = ly.n;
  const int jlast = ((n - 1) >> 2) << 2;
  for (int j = jlast; j >= 0; j -= 4) {
    const int nb = n - j < 4 ? n - j : 4;
    real t[4][4], x[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int c = 0; c < 4; ++c) t[r][c] = (r < nb && c < r) ? s.H[tri(j + r, j + c)] : 0.0;
      x[r] = r < nb ? s.b[j + r] : 0.0;
    }
#pragma unroll
    for (int r = 3; r >= 0; --r) {
      real v = x[r];
#pragma unroll
      for (int k = r + 1; k < 4; ++k) v -= t[k][r] * x[k];
      x[r] = v * (r < nb ? s.d[j + r] : 1.0);   // s.d holds 1 / L_jj (ref_cholesky)
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) if (tid == r && r < nb) s.b[j + r] = x[r];
    for (int k = tid; k < j; k += NT) {
      real acc = 0.0;
#pragma unroll
      for (int r = 0; r < 4; ++r)
        if (r < nb && s.first[j + r] <= k) acc += s.H[tri(j + r, k)] * x[r];
      s.b[k] -= acc;
    }
    __syncthreads();
  }
}

__device__ int ref_update(const Layout& ly, const Ctx& e, const Sm& s, int tid) {
  __shared__ int sh_bad;
  if (tid == 0) sh_bad = 0;
  __syncthreads();
  for (int i = tid; i < ly.n; i += NT) {
    const bool live = i < 3 ? true : (i < 3 * ly.W ? (i / 3) < e.c : (bool)((e.act >> ((i - 3 * ly.W) >> 1)) & 1ull));
    if (!live) continue;
    const real dl = s.b[s.pos[i]];
    if (!isfinite(dl)) sh_bad = 1;
    const real nv = s.v[i] + dl;
    s.v[i] = is_angle(ly, i) ? wrapr(nv) : nv;
  }
  __syncthreads();
  return sh_bad ? slamk::ENV_NONFINITE : 0;
}

// Sigma_t = J Sigma_6 J' from the trailing 6x6 of L (newest pose, anchor), ln det (eq. (6))
__device__ void ref_covariance(const Layout& ly, const Ctx& e, const Sm& s, int tid, const StepIO& io) {
  const int n = ly.n, N = ly.N;
  if (tid == 0) {
    real Lm[6][6], Li[6][6], S6[6][6], T[6][3], S[3][3];
    for (int x = 0; x < 6; ++x)
      for (int y = 0; y < 6; ++y) { Lm[x][y] = y <= x ? s.H[tri(n - 6 + x, n - 6 + y)] : 0.0; Li[x][y] = 0.0; }
    for (int col = 0; col < 6; ++col)
      for (int x = col; x < 6; ++x) {
        real sum = x == col ? 1.0 : 0.0;
        for (int k = col; k < x; ++k) sum -= Lm[x][k] * Li[k][col];
        Li[x][col] = sum / Lm[x][x];
      }
    for (int x = 0; x < 6; ++x)
      for (int y = 0; y < 6; ++y) {
        real sum = 0.0;
        for (int k = (x > y ? x : y); k < 6; ++k) sum += Li[k][x] * Li[k][y];
        S6[x][y] = sum;
      }
    const real ca = cos(s.v[2]), sa = sin(s.v[2]), je = e.c >= 2 ? 1.0 : 0.0;
    const real ex = e.c >= 2 ? s.v[vpose(e.c - 1)] : 0.0, ey = e.c >= 2 ? s.v[vpose(e.c - 1) + 1] : 0.0;
    const real dx = ca * ex - sa * ey, dy = sa * ex + ca * ey;
    const real J[3][6] = {{je * ca, -je * sa, 0, 1, 0, -dy}, {je * sa, je * ca, 0, 0, 1, dx}, {0, 0, je, 0, 0, 1}};
    for (int x = 0; x < 6; ++x)
      for (int j = 0; j < 3; ++j) {
        real sum = 0.0;
        for (int q = 0; q < 6; ++q) sum += S6[x][q] * J[j][q];
        T[x][j] = sum;
      }
    for (int x = 0; x < 3; ++x)
      for (int y = 0; y < 3; ++y) {
        real sum = 0.0;
        for (int q = 0; q < 6; ++q) sum += J[x][q] * T[q][y];
        S[x][y] = sum;
      }
    for (int x = 0; x < 3; ++x)
      for (int y = 0; y < 3; ++y) {
        const float val = (float)(0.5 * (S[x][y] + S[y][x]));
        io.cov_cache[(size_t)(3 * x + y) * N + e.env] = val;
        if (io.cov) io.cov[(size_t)(3 * x + y) * N + e.env] = val;
      }
    const real s01 = 0.5 * (S[0][1] + S[1][0]), s02 = 0.5 * (S[0][2] + S[2][0]), s12 = 0.5 * (S[1][2] + S[2][1]);
    const real det = S[0][0] * (S[1][1] * S[2][2] - s12 * s12) - s01 * (s01 * S[2][2] - s12 * s02) + s02 * (s01 * s12 - S[1][1] * s02);
    const float ld = (float)log(det);
    io.cov_cache[(size_t)9 * N + e.env] = ld;
    if (io.logdet) io.logdet[e.env] = ld;
    if (io.dopt) io.dopt[e.env] = expf(ld * (1.0f / 3.0f));
  }
  __syncthreads();
}

// ------------------------------------------------------------------ marginalise the oldest pose
// Sub-problem on the new support (old prior + factors touching slot 0), congruence with N = E + X P_w',
// Schur complement over w = e_1, new prior written (packed, canonical order) to the record of `newmode`.
__device__ void ref_marginalize(const Layout& ly, const Params& pr, Ctx& e, const Sm& s, int tid, int newmode) {
  const int W = ly.W, L = ly.L, c = e.c;
  int* ri = reinterpret_cast<int*>(e.r32);
  uint32_t* ru = reinterpret_cast<uint32_t*>(e.r32);
  uint64_t lc0 = 0ull;
  for (int k = 1; k < c; ++k) if (s.lct[k] == 0) lc0 |= 1ull << k;
  const uint64_t rb0 = L > 0 ? vis_of(ly, s, 0) : 0ull;
  const uint64_t nps = e.ps | 2ull | lc0, nls = e.ls | rb0;
  const int npn = __popcll(nps), nln = __popcll(nls), npo = __popcll(e.ps);
  const int sn = 3 + 3 * npn + 2 * nln, so = e.s;
  real* Hs = s.H;                      // packed [sn(sn+1)/2]
  real* gam = s.b;                     // [sn]
  // new support position of block (slot k / landmark l)
  auto ppose = [&](int k) { return 3 + 3 * __popcll(nps & lowmask(k)); };
  auto plm = [&](int l) { return 3 + 3 * npn + 2 * __popcll(nls & lowmask(l)); };
  for (int p = tid; p < so; p += NT) {
    real dd = s.v[s.sidx[p]] - ldr(e, ly.o_vbar + p);
    if (is_angle(ly, s.sidx[p])) dd = wrapr(dd);
    s.d[p] = dd;
    int P;
    if (p < 3) P = p;
    else if (p < 3 + 3 * npo) { const int bk = (p - 3) / 3; P = ppose(nth_bit(e.ps, bk)) + (p - 3 - 3 * bk); }
    else { const int q = p - 3 - 3 * npo; P = plm(nth_bit(e.ls, q >> 1)) + (q & 1); }
    s.omap[p] = P;
  }
  for (int t = tid; t < sn * (sn + 1) / 2; t += NT) Hs[t] = 0.0;
  for (int p = tid; p < sn; p += NT) gam[p] = 0.0;
  __syncthreads();
  // old prior: H_s = Lambda, gamma = Lambda d + g
  for (int t = tid; t < so * (so + 1) / 2; t += NT) {
    int p = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((p + 1) * (p + 2) / 2 <= t) ++p;
    while (p * (p + 1) / 2 > t) --p;
    const int q = t - p * (p + 1) / 2;
    Hat(Hs, s.omap[p], s.omap[q]) = ldr(e, ly.o_lam + t);
  }
  __syncthreads();
  for (int p = tid; p < so; p += NT) {
    real acc = ldr(e, ly.o_g + p);
    for (int q = 0; q < so; ++q) acc += Hat(Hs, s.omap[p], s.omap[q]) * s.d[q];
    gam[s.omap[p]] = acc;
  }
  __syncthreads();
  const real sa = sin(s.v[2]), ca = cos(s.v[2]);
  const real x1 = s.v[vpose(1)], y1 = s.v[vpose(1) + 1], th1 = s.v[vpose(1) + 2];
  const real s1 = sin(th1), c1 = cos(th1);
  const real ddx = ca * x1 - sa * y1, ddy = sa * x1 + ca * y1;
  // factors touching slot 0 (the frame: J_j = I for between factors), serial in one thread (few of them)
  if (tid == 0) {
    for (int x = 0; x < 3; ++x) {
      real r = s.v[vpose(1) + x] - (real)e.r32[ly.o_zodo + 3 * ring_of(1, e.head, W) + x];
      if (x == 2) r = wrapr(r);
      Hs[tri(3 + x, 3 + x)] += (real)pr.om_odo[x];
      gam[3 + x] += (real)pr.om_odo[x] * r;
    }
    for (int k = 1; k < c; ++k) {
      if (s.lct[k] != 0) continue;
      const int P = ppose(k);
      for (int x = 0; x < 3; ++x) {
        real r = s.v[vpose(k) + x] - (real)e.r32[ly.o_zlc + 3 * ring_of(k, e.head, W) + x];
        if (x == 2) r = wrapr(r);
        Hs[tri(P + x, P + x)] += (real)pr.om_lc[x];
        gam[P + x] += (real)pr.om_lc[x] * r;
      }
    }
    if (e.um & 1ull) {
      const float* o6 = e.r32 + ly.o_omun + 6 * e.head;
      const real O[3][3] = {{o6[0], o6[1], o6[3]}, {o6[1], o6[2], o6[4]}, {o6[3], o6[4], o6[5]}};
      const real res[3] = {s.v[0] - (real)e.r32[ly.o_zun + 3 * e.head], s.v[1] - (real)e.r32[ly.o_zun + 3 * e.head + 1],
                           wrapr(s.v[2] - (real)e.r32[ly.o_zun + 3 * e.head + 2])};
      for (int x = 0; x < 3; ++x) {
        for (int y = 0; y <= x; ++y) Hs[tri(x, y)] += O[x][y];
        gam[x] += O[x][0] * res[0] + O[x][1] * res[1] + O[x][2] * res[2];
      }
    }
    const real om_rb[2] = {pr.om_rb[0], pr.om_rb[1]};
    for (uint64_t m = rb0; m;) {
      const int l = __ffsll((long long)m) - 1;
      m &= m - 1;
      const Rb f = rangebearing(s.v, ca, sa, s.v, true, s.v + vlm(ly, l), (real)e.r32[ly.o_zrb + (e.head * 2 + 0) * L + l],
                                (real)e.r32[ly.o_zrb + (e.head * 2 + 1) * L + l]);
      const int P = plm(l);
      for (int x = 0; x < 2; ++x) {
        for (int y = 0; y <= x; ++y) Hs[tri(P + x, P + y)] += f.Jg[0][x] * om_rb[0] * f.Jg[0][y] + f.Jg[1][x] * om_rb[1] * f.Jg[1][y];
        for (int y = 0; y < 3; ++y) Hs[tri(P + x, y)] += f.Jg[0][x] * om_rb[0] * f.Ja[0][y] + f.Jg[1][x] * om_rb[1] * f.Ja[1][y];
        gam[P + x] += f.Jg[0][x] * om_rb[0] * f.r[0] + f.Jg[1][x] * om_rb[1] * f.r[1];
      }
      for (int x = 0; x < 3; ++x) {
        for (int y = 0; y <= x; ++y) Hs[tri(x, y)] += f.Ja[0][x] * om_rb[0] * f.Ja[0][y] + f.Ja[1][x] * om_rb[1] * f.Ja[1][y];
        gam[x] += f.Ja[0][x] * om_rb[0] * f.r[0] + f.Ja[1][x] * om_rb[1] * f.r[1];
      }
    }
  }
  // X = N[:, w] - E[:, w] rows (step 3): a: da/dw, e_1: 0, e_k: de_k/dw, landmarks: 0;  new state-index table
  for (int p = tid; p < sn; p += NT) {
    int id;
    real X0 = 0.0, X1 = 0.0, X2 = 0.0;
    if (p < 3) {
      id = p;
      X0 = p == 0 ? -ca : (p == 1 ? -sa : 0.0);
      X1 = p == 0 ? sa : (p == 1 ? -ca : 0.0);
      X2 = p == 0 ? -ddy : (p == 1 ? ddx : -1.0);
    } else if (p < 3 + 3 * npn) {
      const int bk = (p - 3) / 3, j = p - 3 - 3 * bk, k = nth_bit(nps, bk);
      id = vpose(k) + j;
      if (k != 1) {
        X0 = j == 0 ? 1.0 : 0.0; X1 = j == 1 ? 1.0 : 0.0;
        X2 = j == 0 ? -(s.v[vpose(k) + 1] - y1) : (j == 1 ? (s.v[vpose(k)] - x1) : 1.0);
      }
    } else {
      const int q = p - 3 - 3 * npn;
      id = vlm(ly, nth_bit(nls, q >> 1)) + (q & 1);
    }
    s.sidx[p] = id;   // (the old table is dead: d and omap are built)
    s.X[3 * p] = X0; s.X[3 * p + 1] = X1; s.X[3 * p + 2] = X2;
  }
  __syncthreads();
  // Q = H_s X
  for (int p = tid; p < sn; p += NT) {
    real q0 = 0.0, q1 = 0.0, q2 = 0.0;
    for (int q = 0; q < sn; ++q) {
      const real h = Hat(Hs, p, q);
      q0 += h * s.X[3 * q]; q1 += h * s.X[3 * q + 1]; q2 += h * s.X[3 * q + 2];
    }
    s.Q[3 * p] = q0; s.Q[3 * p + 1] = q1; s.Q[3 * p + 2] = q2;
  }
  __syncthreads();
  // Y = X'Q, gx = X'gamma (every thread, serially: 12 sums of length sn)
  real Y[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, gx[3] = {0, 0, 0};
  for (int p = 0; p < sn; ++p)
    for (int x = 0; x < 3; ++x) {
      const real xv = s.X[3 * p + x];
      if (xv == 0.0) continue;
      for (int y = 0; y < 3; ++y) Y[x][y] += xv * s.Q[3 * p + y];
      gx[x] += xv * gam[p];
    }
  __syncthreads();
  // G = E' H_s E in place, block pair by block pair; E_b = [[p,-q,u],[q,p,v],[0,0,1]] (2x2 leading part for landmarks)
  const int nbk = 1 + npn + nln;
  auto bpos = [&](int bk) { return bk == 0 ? 0 : (bk <= npn ? 3 + 3 * (bk - 1) : 3 + 3 * npn + 2 * (bk - 1 - npn)); };
  auto etype = [&](int bk, real* E4) {
    if (bk == 0) { E4[0] = 1.0; E4[1] = 0.0; E4[2] = ddy; E4[3] = -ddx; }                 // da/da'
    else if (bk == 1 || bk > npn) { E4[0] = 1.0; E4[1] = 0.0; E4[2] = 0.0; E4[3] = 0.0; }  // w, landmarks: identity
    else { E4[0] = c1; E4[1] = s1; E4[2] = 0.0; E4[3] = 0.0; }                            // blockdiag(Rot(th_1), 1)
  };
  for (int t = tid; t < nbk * (nbk + 1) / 2; t += NT) {
    int bi = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((bi + 1) * (bi + 2) / 2 <= t) ++bi;
    while (bi * (bi + 1) / 2 > t) --bi;
    const int bj = t - bi * (bi + 1) / 2;
    const int pi = bpos(bi), pj = bpos(bj), di = bi <= npn ? 3 : 2, dj = bj <= npn ? 3 : 2;
    real Ei[4], Ej[4];
    etype(bi, Ei); etype(bj, Ej);
    real M[3][3], T[3][3];
    for (int x = 0; x < 3; ++x)
      for (int y = 0; y < 3; ++y) M[x][y] = (x < di && y < dj) ? Hat(Hs, pi + x, pj + y) : 0.0;
    for (int x = 0; x < 3; ++x) {
      T[x][0] = M[x][0] * Ej[0] + M[x][1] * Ej[1];
      T[x][1] = -M[x][0] * Ej[1] + M[x][1] * Ej[0];
      T[x][2] = M[x][0] * Ej[2] + M[x][1] * Ej[3] + M[x][2];
    }
    for (int y = 0; y < 3; ++y) {
      M[0][y] = Ei[0] * T[0][y] + Ei[1] * T[1][y];
      M[1][y] = -Ei[1] * T[0][y] + Ei[0] * T[1][y];
      M[2][y] = Ei[2] * T[0][y] + Ei[3] * T[1][y] + T[2][y];
    }
    for (int x = 0; x < di; ++x)
      for (int y = 0; y < dj; ++y)
        if (bi != bj || y <= x) Hs[tri(pi + x, pj + y)] = M[x][y];
  }
  __syncthreads();
  // T_b = E_b' Q_b, gamma_b = E_b' gamma_b
  for (int bk = tid; bk < nbk; bk += NT) {
    const int pb = bpos(bk), db = bk <= npn ? 3 : 2;
    real E4[4];
    etype(bk, E4);
    real t0[3], t1[3], t2[3] = {0, 0, 0};
    for (int y = 0; y < 3; ++y) { t0[y] = s.Q[3 * pb + y]; t1[y] = s.Q[3 * (pb + 1) + y]; if (db == 3) t2[y] = s.Q[3 * (pb + 2) + y]; }
    const real g0 = gam[pb], g1 = gam[pb + 1], g2 = db == 3 ? gam[pb + 2] : 0.0;
    for (int y = 0; y < 3; ++y) {
      s.Q[3 * pb + y] = E4[0] * t0[y] + E4[1] * t1[y];
      s.Q[3 * (pb + 1) + y] = -E4[1] * t0[y] + E4[0] * t1[y];
      if (db == 3) s.Q[3 * (pb + 2) + y] = E4[2] * t0[y] + E4[3] * t1[y] + t2[y];
    }
    gam[pb] = E4[0] * g0 + E4[1] * g1;
    gam[pb + 1] = -E4[1] * g0 + E4[0] * g1;
    if (db == 3) gam[pb + 2] = E4[2] * g0 + E4[3] * g1 + g2;
  }
  __syncthreads();
  // H_ww, gamma_w; K = G[:, w] + T; KW = K H_ww^{-1}
  real Hw[3][3], gw[3], Wi[3][3];
  for (int x = 0; x < 3; ++x) {
    gw[x] = gam[3 + x] + gx[x];
    for (int y = 0; y < 3; ++y) Hw[x][y] = Hat(Hs, 3 + x, 3 + y) + s.Q[3 * (3 + x) + y] + s.Q[3 * (3 + y) + x] + Y[x][y];
  }
  {
    const real c00 = Hw[1][1] * Hw[2][2] - Hw[1][2] * Hw[2][1], c01 = Hw[1][2] * Hw[2][0] - Hw[1][0] * Hw[2][2];
    const real c02 = Hw[1][0] * Hw[2][1] - Hw[1][1] * Hw[2][0];
    const real id = 1.0 / (Hw[0][0] * c00 + Hw[0][1] * c01 + Hw[0][2] * c02);
    Wi[0][0] = c00 * id; Wi[1][0] = c01 * id; Wi[2][0] = c02 * id;
    Wi[0][1] = (Hw[0][2] * Hw[2][1] - Hw[0][1] * Hw[2][2]) * id;
    Wi[1][1] = (Hw[0][0] * Hw[2][2] - Hw[0][2] * Hw[2][0]) * id;
    Wi[2][1] = (Hw[0][1] * Hw[2][0] - Hw[0][0] * Hw[2][1]) * id;
    Wi[0][2] = (Hw[0][1] * Hw[1][2] - Hw[0][2] * Hw[1][1]) * id;
    Wi[1][2] = (Hw[0][2] * Hw[1][0] - Hw[0][0] * Hw[1][2]) * id;
    Wi[2][2] = (Hw[0][0] * Hw[1][1] - Hw[0][1] * Hw[1][0]) * id;
  }
  __syncthreads();
  for (int r = tid; r < sn; r += NT) {
    if (r >= 3 && r < 6) continue;
    real K[3];
    for (int y = 0; y < 3; ++y) K[y] = s.Q[3 * r + y] + Hat(Hs, r, 3 + y);
    for (int y = 0; y < 3; ++y) {
      s.Q[3 * r + y] = K[y];
      s.X[3 * r + y] = K[0] * Wi[0][y] + K[1] * Wi[1][y] + K[2] * Wi[2][y];
    }
  }
  __syncthreads();
  // new state: a <- a (+) e_1, e_k <- between(e_1, e_k), slot 1 becomes the frame
  for (int k = 2 + tid; k < c; k += NT) {
    real* q = s.v + vpose(k);
    const real ex = q[0] - x1, ey = q[1] - y1;
    q[0] = c1 * ex + s1 * ey; q[1] = -s1 * ex + c1 * ey; q[2] = wrapr(q[2] - th1);
  }
  __syncthreads();
  if (tid == 0) { s.v[0] += ddx; s.v[1] += ddy; s.v[2] = wrapr(s.v[2] + th1); }
  if (tid < 3) s.v[vpose(1) + tid] = 0.0;
  __syncthreads();
  // new prior on the support without w
  float* o32 = e.r32;
  double* o64 = e.r64;
  for (int t = tid; t < sn * (sn + 1) / 2; t += NT) {
    int r = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((r + 1) * (r + 2) / 2 <= t) ++r;
    while (r * (r + 1) / 2 > t) --r;
    const int q = t - r * (r + 1) / 2;
    if ((r >= 3 && r < 6) || (q >= 3 && q < 6)) continue;
    const int R = r < 3 ? r : r - 3, Qn = q < 3 ? q : q - 3;
    const real val = Hs[t] - (s.X[3 * r] * s.Q[3 * q] + s.X[3 * r + 1] * s.Q[3 * q + 1] + s.X[3 * r + 2] * s.Q[3 * q + 2]);
    if (newmode) o64[ly.o_lam + tri(R, Qn)] = val; else o32[ly.o_lam + tri(R, Qn)] = (float)val;
  }
  for (int r = tid; r < sn; r += NT) {
    if (r >= 3 && r < 6) continue;
    const int R = r < 3 ? r : r - 3;
    const real gv = gam[r] - (s.X[3 * r] * gw[0] + s.X[3 * r + 1] * gw[1] + s.X[3 * r + 2] * gw[2]);
    const real vb = s.v[s.sidx[r]];
    if (newmode) { o64[ly.o_g + R] = gv; o64[ly.o_vbar + R] = vb; } else { o32[ly.o_g + R] = (float)gv; o32[ly.o_vbar + R] = (float)vb; }
  }
  for (int k = 1 + tid; k < c; k += NT)
    if (s.lct[k] == 0) ri[ly.o_lct + ring_of(k, e.head, W)] = -1;
  e.um &= ~1ull;
  e.ps = nps & ~2ull;
  e.ls = nls;
  if (tid == 0) {
    const uint64_t pm = slot_to_ring(e.ps, e.head, W);
    ru[ly.o_pm] = (uint32_t)pm; ru[ly.o_pm + 1] = (uint32_t)(pm >> 32);
    ru[ly.o_lm] = (uint32_t)nls; ru[ly.o_lm + 1] = (uint32_t)(nls >> 32);
  }
  __syncthreads();
}

// state (a, e at the ring positions of the current head, landmarks, masks) into the record of `newmode`;
// without a marginalisation in this call the prior moves along when the mode changes
__device__ void ref_store(const Layout& ly, const Ctx& e, const Sm& s, int tid, int newmode, bool prior_written) {
  const int W = ly.W, L = ly.L;
  uint32_t* ru = reinterpret_cast<uint32_t*>(e.r32);
  auto put = [&](int off, real val) { if (newmode) e.r64[off] = val; else e.r32[off] = (float)val; };
  if (tid < 3) put(ly.o_a + tid, s.v[tid]);
  for (int i = 3 + tid; i < 3 * e.c; i += NT) { const int k = i / 3; put(ly.o_e + 3 * ring_of(k, e.head, W) + (i - 3 * k), s.v[i]); }
  if (tid < 3) put(ly.o_e + 3 * ring_of(0, e.head, W) + tid, 0.0);
  for (int i = tid; i < 2 * L; i += NT) put(ly.o_m + i, s.v[3 * W + i]);
  if (newmode != e.mode && !prior_written) {
    const int so = 3 + 3 * __popcll(e.ps) + 2 * __popcll(e.ls);
    for (int t = tid; t < so * (so + 1) / 2; t += NT) put(ly.o_lam + t, ldr(e, ly.o_lam + t));
    for (int p = tid; p < so; p += NT) { put(ly.o_g + p, ldr(e, ly.o_g + p)); put(ly.o_vbar + p, ldr(e, ly.o_vbar + p)); }
  }
  if (tid == 0) {
    ru[ly.o_act] = (uint32_t)e.act; ru[ly.o_act + 1] = (uint32_t)(e.act >> 32);
    const uint64_t um = slot_to_ring(e.um, e.head, W);
    ru[ly.o_um] = (uint32_t)um; ru[ly.o_um + 1] = (uint32_t)(um >> 32);
    reinterpret_cast<int*>(e.r32)[ly.o_mode] = newmode;
  }
}

// ------------------------------------------------------------------ the kernel: persistent CTAs pull environments from the list
__global__ void __launch_bounds__(NT, 4) slam_ref64_kernel(Layout ly, Params pr, RefArgs ra, StepIO io) {
  extern __shared__ double ref_smem[];
  __shared__ int sh_i;
  const int tid = threadIdx.x;
  double* hglob = ra.hglob ? ra.hglob + (size_t)blockIdx.x * ref_tri(ly) : nullptr;
  const Sm s = carve(ly, ref_smem, hglob);
  const int nlin = ra.iters + ((ra.flags & slamk::F_COV) ? 1 : 0);
  for (;;) {
    __syncthreads();
    if (tid == 0) sh_i = atomicAdd(ra.cnt + 1, 1);
    __syncthreads();
    const int i = sh_i;
    if (i >= ra.cnt[0]) break;
    Ctx e;
    e.env = ra.list[i];
    e.r32 = ra.state32 + (size_t)e.env * ly.rec;
    e.r64 = ra.state64 + (size_t)e.env * ly.rec;
    const int* ri = reinterpret_cast<const int*>(e.r32);
    e.k0 = ri[ly.o_k0];
    e.mode = ri[ly.o_mode];
    e.head = (ra.head_g + e.k0) % ly.W;
    e.c = ra.c - e.k0;
    ref_load(ly, e, s, tid);
    if (ra.flags & slamk::F_OBS0) ref_record_rb(ly, e, s, tid, 0, 0.0, 0.0, 0.0, io);
    if (ra.flags & slamk::F_PUSH) ref_push(ly, e, s, tid, io);
    ref_order(ly, e, s, tid);
    int status = 0;
    real ratio = 0.0;
    __shared__ real sh_ratio;
    if (tid == 0) sh_ratio = 0.0;
    __syncthreads();
    for (int it = 0; it < nlin; ++it) {
      ref_assemble(ly, pr, e, s, tid);
      { REF_TICK_DECL status |= ref_cholesky(ly, s, tid, &sh_ratio); REF_TICK(6) }
      if (it < ra.iters) {
        ref_backsub(ly, s, tid);
        status |= ref_update(ly, e, s, tid);
      } else {
        ref_covariance(ly, e, s, tid, io);
      }
    }
    __syncthreads();
    ratio = sh_ratio;
    if (io.last_pose && tid == 0) {
      const real sn = sin(s.v[2]), cn = cos(s.v[2]);
      const real ex = e.c >= 2 ? s.v[vpose(e.c - 1)] : 0.0, ey = e.c >= 2 ? s.v[vpose(e.c - 1) + 1] : 0.0, et = e.c >= 2 ? s.v[vpose(e.c - 1) + 2] : 0.0;
      io.last_pose[e.env] = (float)(s.v[0] + cn * ex - sn * ey);
      io.last_pose[(size_t)ly.N + e.env] = (float)(s.v[1] + sn * ex + cn * ey);
      io.last_pose[2 * (size_t)ly.N + e.env] = (float)wrapr(s.v[2] + et);
    }
    // precision mode of the record after this call: fp64 while the anchor pivots cancel, back to fp32 below ratio_lo
    int newmode = e.mode;
    // Back to fp32 only while the robot is localised against the map: the newest pose must see at least `min_vis`
    // landmarks.  A robot that leaves the map right after the hand-over dead-reckons on a prior whose landmark and
    // anchor blocks still carry the cancellation of the ill-conditioned phase; fp32 marginalisations lose it within
    // tens of steps although the anchor pivots look harmless (measured: 18 of the 21 env-steps beyond tolerance of a
    // 4096-environment sample of config 3).
    if (nlin > 0) {
      const int nvis = ly.L > 0 ? __popcll(vis_of(ly, s, e.c - 1)) : 0;
      const bool well = ly.L > 0 && ra.box_vis > 0 && nvis >= ra.box_vis;   // well localised: twice the threshold, as in slam_step_kernel
      newmode = (ratio < (well ? 2.0 : 1.0) * ra.ratio_lo && status == 0 && (ly.L == 0 || nvis >= ra.min_vis)) ? 0 : 1;
    }
    if (ra.force) newmode = 1;
    const bool do_marg = (ra.flags & slamk::F_MARG) && e.k0 == 0;
    if (do_marg) ref_marginalize(ly, pr, e, s, tid, newmode);
    else if ((ra.flags & slamk::F_MARG) && tid == 0) reinterpret_cast<int*>(e.r32)[ly.o_k0] = e.k0 - 1;
    ref_store(ly, e, s, tid, newmode, do_marg);
    if (tid == 0) {
      if (status) atomicOr(reinterpret_cast<int*>(e.r32) + ly.o_status, status);
      if (ra.stats) atomicAdd(ra.stats + 4, 1ull);
      // An environment that stays here costs the step kernel nothing: key 0 sorts it to the END of the cost-ordered
      // list, so the teams that draw it (they only pass it on to this kernel and idle for the round) do so in the
      // last rounds of a launch instead of leaving holes in every round.  One that goes back gets a middling key
      // for one step.
      if (ra.keys) ra.keys[e.env] = newmode ? 0 : ly.dense / 3;
    }
  }
  // the last CTA to leave resets the list for the next launch
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    if (atomicAdd(ra.cnt + 2, 1) == (int)gridDim.x - 1) { ra.cnt[0] = 0; ra.cnt[1] = 0; ra.cnt[2] = 0; }
  }
}

}  // namespace slamr
