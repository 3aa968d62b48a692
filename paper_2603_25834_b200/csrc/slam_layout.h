// Device-memory and shared-memory layout of one environment (host + device).
//
// HBM: one contiguous, 16-byte aligned RECORD per environment ("array of per-environment
// structures of arrays"), so that the warp that owns an environment reads and writes coalesced,
// contiguous runs and the whole record can be staged by bulk copies.  Slot arrays are RING BUFFERS
// indexed by ring position r = (head + slot) % W: marginalisation advances `head` and never moves
// factor data (north_star "ring-buffer window shift").
//
// The marginalisation prior is stored on its SUPPORT only: two 64-bit masks (pose ring positions,
// landmarks) name the support blocks in canonical order [anchor a | poses by ascending slot |
// landmarks by ascending index]; Lambda is packed lower-triangular over that order.
#pragma once
#include <stdint.h>

namespace slamk {

struct Layout {
  int N, W, L, n, nw;  // n = 3W + 2L state dimension, nw = ceil(L/32) mask words
  int np, pad;         // matrix dimension padded to a multiple of 4 (pad dummy rows before the newest pose)
  // record (32-bit words)
  int rec;             // record stride
  int o_status, o_k0, o_pm, o_lm, o_act, o_um, o_mode, o_a, o_e, o_m, o_zodo, o_lct, o_zlc, o_rbm, o_zrb, o_zun, o_omun, o_vbar, o_g, o_lam;
  // shared memory: a FIXED part per team (32-bit words) ...
  int s_scr, s_st, s_lct, s_cs, s_rbm, s_rbf, s_sup, s_sds;
  int team_words;      // fixed shared words per team
  // ... and one POOL per CTA from which every environment of a round takes what its envelope needs
  // (H + rhs rows + active-pair lists, or the marginalisation scratch): slam_step_kernel
  int pool;            // words of the pool (>= dense: one environment always fits)
  int cap;             // = pool: the most one environment can get
  int dense;           // words that suffice for ANY environment of this size
  int wpc;             // teams (environments in flight) per CTA
  int team;            // threads per environment: 32, 64 or 128
  int pairs;           // 1: envelope rows grouped in pairs instead of fours (less shared memory, more instructions)
  int lcache;          // 1: keep the factor columns of passive landmarks across the linearisations of one call
  int pf_bytes;        // bytes of the next round's record pulled into L2 by cp.async.bulk.prefetch (0: off)
  int dynq;            // 1: the CTAs take their chunks of the ordered list from one queue for the grid
  int lock;            // lock-step level: CTA barriers before assemble (1), + before Cholesky (2), + before the solve (3)
  int box_vis;         // landmarks the newest pose must see to count as well localised (doubles the thresholds of the watch; 0: off)
  float ratio_hi;      // anchor pivot ratio H_aa / L_aa^2 above which the fp32 kernel hands the environment to the fp64 path (0: never)
};

struct Params {
  float om_prior[3], om_odo[3], om_lc[3], om_rb[2];  // information = 1 / sigma^2
};

static inline int pad4(int x) { return (x + 3) & ~3; }

// Fills every offset.  `pool` = words of the CTA pool (raised to the dense need of one environment).
static inline Layout make_layout(int N, int W, int L, int pool, int wpc) {
  Layout y;
  y.N = N; y.W = W; y.L = L; y.n = 3 * W + 2 * L; y.nw = (L + 31) / 32;
  y.np = (y.n + 3) & ~3; y.pad = y.np - y.n;
  int n = y.n, o = 0;
  y.o_status = o; o += 1;
  y.o_k0 = o; o += 1;   // NEXT-2: first live slot of this environment (0 unless it was reset mid-run)
  y.o_pm = o; o += 2;
  y.o_lm = o; o += 2;
  y.o_act = o; o += 2;
  y.o_um = o; o += 2;   // ring positions that carry a unary absolute-pose factor
  y.o_mode = o; o += 1; // 0: state and prior live in this fp32 record; 1: in the fp64 shadow record (slam_ref64.cuh)
  o = pad4(o + 1);
  y.o_a = o; o += 4;
  y.o_e = o; o = pad4(o + 3 * W);
  y.o_m = o; o = pad4(o + 2 * L);
  y.o_zodo = o; o = pad4(o + 3 * W);
  y.o_lct = o; o = pad4(o + W);
  y.o_zlc = o; o = pad4(o + 3 * W);
  y.o_rbm = o; o = pad4(o + W * y.nw);
  y.o_zrb = o; o = pad4(o + W * 2 * L);
  y.o_zun = o; o = pad4(o + 3 * W);    // unary factors: measured global pose per ring position
  y.o_omun = o; o = pad4(o + 6 * W);   // ... and its information (xx, xy, yy, xt, yt, tt)
  y.o_vbar = o; o = pad4(o + n);
  y.o_g = o; o = pad4(o + n);
  y.o_lam = o; o = pad4(o + n * (n + 1) / 2);
  y.rec = (o + 31) & ~31;  // 128-byte multiple

  int s = 0;
  y.s_scr = s; s += 64;   // team scratch (reductions, diagonal tile, counters)
  y.s_st = s; s = pad4(s + n + 3);
  y.s_lct = s; s = pad4(s + W + 2);  // + the loop-closure mask (two words)
  y.s_cs = s; s = pad4(s + 2 * W);
  y.s_rbm = s; s = pad4(s + W * y.nw);
  y.s_rbf = s; s = pad4(s + y.np + 2);   // row pointer | first column, packed
  y.s_sup = s; s = pad4(s + n);          // prior support: elimination offset | state index, packed
  // prior displacement (<= n) + anchor-frame landmarks (2L); scratch of the symbolic phase (np + 2)
  y.s_sds = s; s = pad4(s + (n + 2 * L > y.np + 2 ? n + 2 * L : y.np + 2));
  y.team_words = pad4(s);
  // dense need of one environment: full 4x4 tiles of the lower triangle + the rhs row + the tables of
  // the factorisation (G+1 column headers, NP row-pair entries, at most sum_J (NP - 2J) pair indices of 8 bit);
  // or the marginalisation scratch; or the fp64 scratch of the covariance tail
  const int G = y.np / 4, NPp = y.np / 2 + 1;
  const int list_bytes = G * NPp - G * (G - 1);
  int dense = 8 * G * (G + 1) + y.np + pad4((G + 1) + NPp + (list_bytes + 3) / 4);
  const int marg = n * (n + 1) / 2 + 8 * n + 16;
  if (marg > dense) dense = marg;
  if (dense < 272) dense = 272;
  y.dense = pad4(dense);
  y.pool = pool < y.dense ? y.dense : (pool & ~3);
  y.cap = y.pool;
  y.wpc = wpc;
  y.team = 32;
  y.lock = 1;
  y.dynq = 0;
  y.pf_bytes = 0;
  y.ratio_hi = 0.f;
  y.box_vis = 0;
  y.lcache = 1;
  y.pairs = 0;
  return y;
}

}  // namespace slamk
