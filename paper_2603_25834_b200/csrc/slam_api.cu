// C ABI of the batched fixed-lag SLAM backbone (include/slam.h): host dispatcher + kernels.
// Every step of the hot path runs in the kernels of slam_kernels.cuh; this file only checks
// arguments, keeps the lock-step window bookkeeping (count, ring head) and launches.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/slam.h"
#include "slam_kernels.cuh"
#include "slam_ref64.cuh"

using namespace slamk;

// ------------------------------------------------------------------ kernels
// One TEAM of 32/64/128 threads per environment, `wpc` teams per CTA, persistent CTAs that take their environments
// from one queue over the cost-ordered list (see the assignment below) in ROUNDS.  flags select the phases, so that the
// separate ABI calls and the fused slam_step share the same device code and are bit-for-bit identical.
//
// Shared memory = a fixed part per team (state, factor data, row tables) + ONE POOL per CTA.  The
// envelope of H is data dependent (a third to all of the dense size), so a fixed dense slot per team
// would leave most of the shared memory unused.  Instead, in every round each team loads its
// environment, runs the symbolic phase to learn how many words it NEEDS (envelope + rhs rows +
// active-pair lists, or the marginalisation scratch), and the pool is handed out first-fit in team
// order; a team that does not fit keeps its environment (loaded, untouched in memory) and goes FIRST in
// the next round.  The pool is at least the dense need, so a waiting team always gets in.  Which round
// solves an environment does not change a single bit of its result.
#ifndef SLAM_MAXTHREADS
#define SLAM_MAXTHREADS 512
#endif
template <int TEAM, bool PAIRS, bool LM>
__global__ void __launch_bounds__(TEAM == 128 ? 896 : SLAM_MAXTHREADS)
slam_step_kernel(Layout ly, Params pr, float* state, int head_g, int c, int flags, int iters, StepIO io,
                 unsigned long long* stats, const int* __restrict__ perm, int* __restrict__ keys,
                 int* __restrict__ fb_list, int* __restrict__ fb_cnt) {
  extern __shared__ float4 smem4[];
  __shared__ int s_env[16], s_need[16], s_off[16], s_new[16], s_nxt[16], s_ctl[3];
  int* queue = reinterpret_cast<int*>(stats + 16);   // [0] next entry of the cost-ordered list (ly.dynq), [1] CTAs finished
  float* smem = reinterpret_cast<float*>(smem4);
  const int team = threadIdx.x / TEAM, lane = threadIdx.x % TEAM;
  const int LOCK = ly.lock;
  float* base = smem + (size_t)team * ly.team_words;
  float* pool = smem + (size_t)ly.wpc * ly.team_words;
  WS w = make_ws(ly, base);
  Team<TEAM> tm;
  tm.bar = 1 + team;
  tm.scr = base + ly.s_scr;
  Team<32> tm32;
  tm32.bar = 0;
  tm32.scr = tm.scr;
  // The warp of a team that works alone in the single-warp phases.  Warps are spread over the four
  // sub-partitions of the SM by warp index mod 4: with two warps per team and always the first one working,
  // only sub-partitions 0 and 2 would issue (measured: "not selected" stalls 19 % while two sub-partitions
  // idle), so teams alternate.
  const int solo = TEAM == 64 ? ((team >> 1) & 1) : 0;
  // iters Gauss-Newton iterations, then (F_COV) one more linearisation + factorisation at the final
  // estimate for the covariance: ONE call site per phase keeps the kernel small.
  const int nlin = iters + ((flags & F_COV) ? 1 : 0);
  // the environment this team has in hand (kept across rounds while it waits for pool space)
  int env = -1, k0 = 0, head = 0, cc = 0, s = 0, total = 0, need = 0;
  float rhi = 0.f;   // this environment's threshold of the conditioning watch
  bool waiting = false, do_marg = false;
  Masks mk;
  Ord od;
  if (threadIdx.x < 16) { s_env[threadIdx.x] = -1; s_off[threadIdx.x] = 0; }
  if (threadIdx.x == 0) { s_ctl[0] = 0; s_ctl[2] = 0; }
  // All teams of a CTA walk through the phases in LOCK-STEP (CTA barriers between phases): the kernel is
  // large (~12 k instructions) and instruction-fetch bound, so warps that execute the same code at the
  // same time share every fetched line.  Teams without an environment only take part in the barriers.
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) {  // teams that are not waiting take the next environments, in team order
      int nk = s_ctl[0], live = 0;
      // ly.dynq: the teams of this round take CONSECUTIVE entries of the cost-ordered list (slam_order_kernel) from
      // ONE queue for the whole grid -- the environments of one round cost about the same, so the lock-step
      // barriers wait for little, and a CTA whose teams had to wait for pool space simply takes fewer: no CTA is
      // left with rounds to run after the others have finished (measured: step kernel -4 % against the static deal,
      // SLAM_DYNQ=0: chunks of wpc consecutive entries dealt round-robin to the CTAs)
      int qbase = ly.N;
      if (ly.dynq && s_ctl[2] >= 0) {
        int nfree = 0;
        for (int t = 0; t < ly.wpc; ++t) nfree += s_off[t] != -1;
        if (nfree > 0) {
          qbase = atomicAdd(queue, nfree);
          if (qbase >= ly.N) { s_ctl[2] = -1; qbase = ly.N; }   // the list is exhausted: no more trips to the queue
        }
      }
      for (int t = 0; t < ly.wpc; ++t) {
        if (s_off[t] != -1) {
          const int idx = ly.dynq ? qbase++ : ((nk / ly.wpc) * (int)gridDim.x + (int)blockIdx.x) * ly.wpc + nk % ly.wpc;
          if (idx < ly.N) { s_env[t] = perm[idx]; ++nk; } else s_env[t] = -1;
        }
        live += s_env[t] >= 0;
      }
      s_ctl[0] = nk; s_ctl[1] = live;
      // the environments of the NEXT round (if no team has to wait for pool space), for the L2 prefetch experiment
      if (ly.pf_bytes > 0 && !ly.dynq)
        for (int t = 0; t < ly.wpc; ++t, ++nk) {
          const int idx = ((nk / ly.wpc) * (int)gridDim.x + (int)blockIdx.x) * ly.wpc + nk % ly.wpc;
          s_nxt[t] = idx < ly.N ? perm[idx] : -1;
        }
    }
    __syncthreads();
    if (s_ctl[1] == 0) break;
    // Staging of the next environments' factors (north_star (c); an experiment switch, off by default): ONE
    // cp.async.bulk.prefetch.L2 per team brings the live part of the next record (state, masks, measurements, prior
    // mean / gradient and the head of the packed Lambda) from HBM into L2 a whole round (~0.3 ms) before load_env /
    // assemble touch it.  Not staged into shared memory: every KB of it is pool space, i.e. environments in flight
    // (DESIGN.md section 12 has the measurement).
    if (ly.pf_bytes > 0 && lane == 0 && s_nxt[team] >= 0) {
      const float* nrec = state + (size_t)s_nxt[team] * ly.rec;
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nrec), "r"(ly.pf_bytes) : "memory");
    }
    if (!waiting) {
      env = s_env[team];
      // an environment whose state and prior live in the fp64 shadow record belongs to the fp64 path
      // (slam_ref64.cuh): queue it there and leave this team idle for the round
      if (env >= 0 && fb_list && reinterpret_cast<const int*>(state + (size_t)env * ly.rec)[ly.o_mode] != 0) {
        if (lane == 0) { fb_list[atomicAdd(fb_cnt, 1)] = env; s_env[team] = -1; }
        env = -1;
      }
      if (env >= 0) {
        float* rec = state + (size_t)env * ly.rec;
        // NEXT-2: an environment that was reset mid-run lives in the slots k0.. of the lock-step window:
        // its own count is c - k0 and its ring head is head + k0 (slam_reset_envs).
        k0 = reinterpret_cast<const int*>(rec)[ly.o_k0];
        head = (head_g + k0) % ly.W;
        cc = c - k0;
        load_env<TEAM>(ly, rec, w, tm, lane, head, cc, mk);
        if (flags & F_OBS0) record_rb<TEAM>(ly, rec, w, tm, lane, env, head, 0, 0.f, 0.f, 0.f, io, mk);
        if (flags & F_PUSH) cc = push_env<TEAM>(ly, rec, w, tm, lane, env, head, cc, io, mk);
        od = make_ord(ly, w.rbm, cc);
        // A robot that is WELL localised against the map (its newest pose sees at least box_vis landmarks) gets twice
        // the thresholds of the conditioning watch: with that many fresh measurements per step the result hardly
        // leans on the prior, so what fp32 loses in the anchor's pivots does not accumulate.
        rhi = ly.ratio_hi;
        if (LM && ly.box_vis > 0) {
          int nv = __popc(w.rbm[(cc - 1) * ly.nw]);
          if (ly.nw > 1) nv += __popc(w.rbm[(cc - 1) * ly.nw + 1]);
          if (nv >= ly.box_vis) rhi *= 2.f;
        }
        s = build_support<TEAM>(ly, od, w, tm, lane, cc, mk.ps, mk.ls);
        do_marg = (flags & F_MARG) && k0 == 0;   // a reset environment is not full yet
        need = do_marg ? marg_need(ly, w, lane, cc, mk) : 0;
        total = 0;
        if (nlin > 0) {
          total = symbolic<TEAM>(ly, od, w, tm, lane, cc, mk, s);
          need = max(need, total + reinterpret_cast<const int*>(tm.scr)[10]);
          if (flags & F_COV) need = max(need, 272);  // fp64 scratch of the covariance tail
          if (lane == 0) keys[env] = total;  // cost key for the order of the next launches
          if (stats && lane == 0) {  // envelope statistics (words per environment): max, sum, count
            atomicMax(stats + 0, (unsigned long long)total);
            atomicAdd(stats + 1, (unsigned long long)total);
            atomicAdd(stats + 2, 1ull);
          }
        }
        need = (need + 3) & ~3;
      }
    }
    if (lane == 0) s_need[team] = env >= 0 ? need : 0;
    __syncthreads();
    if (threadIdx.x == 0) {  // first fit in team order, the teams that waited first
      int off = 0;
      for (int pass = 0; pass < 2; ++pass)
        for (int t = 0; t < ly.wpc; ++t) {
          if (s_env[t] < 0) { s_new[t] = 0; continue; }
          if ((s_off[t] == -1) != (pass == 0)) continue;
          const int nd = s_need[t];
          if (nd > ly.pool) s_new[t] = -2;
          else if (off + nd <= ly.pool) { s_new[t] = off; off += nd; }
          else s_new[t] = -1;
        }
      for (int t = 0; t < ly.wpc; ++t) s_off[t] = s_new[t];
    }
    __syncthreads();
    const int off = env >= 0 ? s_off[team] : -3;
    const bool valid = off >= 0;
    waiting = off == -1;
    float* rec = state + (size_t)(env >= 0 ? env : 0) * ly.rec;
    if (lane == 0) {
      if (off == -2) reinterpret_cast<int*>(rec)[ly.o_status] |= 4;  // (cannot happen: the pool holds a dense window)
      if (waiting && stats) atomicAdd(stats + 3, 1ull);
    }
    int status = 0;
    bool single_warp = false;
    if (valid) {
      w.H = pool + off;
      w.amask = reinterpret_cast<uint32_t*>(w.H + total);
      if (nlin > 0) {
        build_lists<TEAM>(ly, w, tm, lane);
        single_warp = reinterpret_cast<const int*>(tm.scr)[9] <= 32;
      }
    }
    if (nlin > 0) {
#pragma unroll 1
      for (int it = 0; it < nlin; ++it) {
        if (LOCK >= 1) __syncthreads();
        // after the first factorisation the column blocks of the passive landmarks keep their factor
        const int ncb = (LM && valid && it > 0 && ly.lcache) ? od.npas >> 1 : 0;
        if (valid) { assemble<TEAM>(ly, pr, od, rec, w, tm, lane, head, cc, mk, s, total, 4 * ncb); tm.sync(); }
        if (LOCK >= 2) __syncthreads();
        if (valid) {
          // When no column block has more than 32 active row pairs (every pose-only window), one warp
          // does the factorisation with shuffles and __syncwarp only: no named barriers, no
          // shared-memory exchange of the diagonal tile.  The other warps of the team wait.
          if (TEAM > 32 && single_warp) {
            if ((lane >> 5) == solo) status |= cholesky<32, PAIRS, LM>(ly, w, tm32, lane & 31, ncb, rhi);
            tm.sync();
          } else {
            status |= cholesky<TEAM, PAIRS, LM>(ly, w, tm, lane, ncb, rhi);
          }
        }
        if (LOCK >= 3) __syncthreads();
        if (valid) {
          if (it < iters) {
            if (TEAM > 32) {  // short rows: one warp, no named barriers
              if ((lane >> 5) == solo) back_substitute<32, PAIRS>(ly, w, tm32, lane & 31);
              tm.sync();
            } else {
              back_substitute<TEAM, PAIRS>(ly, w, tm, lane);
            }
            status |= apply_update<TEAM>(ly, od, w, tm, lane, cc, mk);
          } else {
            covariance<TEAM>(ly, w, tm, lane, env, cc, io);
            tm.sync();
          }
        }
      }
    }
    if (LOCK >= -1) __syncthreads();
    // Conditioning: the anchor pivots cancelled beyond what fp32 can carry (or the
    // factorisation failed outright).  Nothing of this call is committed for the environment -- the record still
    // holds its state before the call -- and the fp64 path redoes the call.
    bool redo = false;
    if (valid && fb_list && nlin > 0) {
      redo = tm.any(status != 0, lane);
      if (redo && lane == 0) fb_list[atomicAdd(fb_cnt, 1)] = env;
    }
    if (valid && !redo) {
      status &= ~ENV_ILLCOND;
      if (io.last_pose && lane == 0) {  // newest pose in global coordinates: a (+) e_{c-1}
        float sn, cn;
        sincos_pi(w.st[2], &sn, &cn);
        const float* e = w.st + st_pose(cc - 1);
        io.last_pose[env] = w.st[0] + cn * e[0] - sn * e[1];
        io.last_pose[(size_t)ly.N + env] = w.st[1] + sn * e[0] + cn * e[1];
        io.last_pose[2 * (size_t)ly.N + env] = wrapf(w.st[2] + e[2]);
      }
      if (do_marg) status |= marginalize<TEAM>(ly, pr, rec, w, tm, lane, head, cc, mk, s);
      else if ((flags & F_MARG) && lane == 0) reinterpret_cast<int*>(rec)[ly.o_k0] = k0 - 1;  // the window slides under it
      store_state<TEAM>(ly, rec, w, tm, lane, head, cc, mk);
      if (status && (lane & 31) == 0) atomicOr(reinterpret_cast<int*>(rec) + ly.o_status, status);  // (any warp may hold a flag)
      tm.sync();
    }
  }
  if (ly.dynq && threadIdx.x == 0) {   // the last CTA to leave rewinds the queue for the next launch
    __threadfence();
    if (atomicAdd(queue + 1, 1) == (int)gridDim.x - 1) { queue[0] = 0; queue[1] = 0; __threadfence(); }
  }
}

// Cost order of the environments for the next launches: counting sort of keys[] (envelope words of the
// last solve, a good predictor of this step's cost: the window slides by one pose) into perm[], most
// expensive first.  One CTA.  Keys cluster (many environments share an envelope size), so lanes with the
// same bucket are combined by __match_any_sync before the shared-memory atomic.  The order inside a
// bucket is arbitrary -- scheduling only, the results do not depend on it.
#define ORDER_BUCKETS 1024
__global__ void __launch_bounds__(1024) slam_order_kernel(int N, int key_max, const int* __restrict__ keys, int* __restrict__ perm) {
  __shared__ int cnt[ORDER_BUCKETS];
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31;
  cnt[tid] = 0;
  __syncthreads();
  const float scale = (float)(ORDER_BUCKETS - 1) / (float)(key_max > 0 ? key_max : 1);
  const int rounds = (N + 1023) >> 10;
  for (int r = 0; r < rounds; ++r) {
    const int i = r * 1024 + tid;
    const int b = i < N ? ORDER_BUCKETS - 1 - (int)((float)min(max(keys[i], 0), key_max) * scale) : -1;
    const unsigned m = __match_any_sync(0xffffffffu, b);
    if (b >= 0 && lane == __ffs(m) - 1) atomicAdd(&cnt[b], __popc(m));
  }
  __syncthreads();
  // exclusive scan of the 1024 counters
  const int v = cnt[tid];
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) wsum[tid >> 5] = x;
  __syncthreads();
  if (tid < 32) {
    int w = wsum[tid];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, w, o); if (tid >= o) w += y; }
    wsum[tid] = w;
  }
  __syncthreads();
  cnt[tid] = x - v + (tid >= 32 ? wsum[(tid >> 5) - 1] : 0);
  __syncthreads();
  for (int r = 0; r < rounds; ++r) {
    const int i = r * 1024 + tid;
    const int b = i < N ? ORDER_BUCKETS - 1 - (int)((float)min(max(keys[i], 0), key_max) * scale) : -1;
    const unsigned m = __match_any_sync(0xffffffffu, b);
    const int leader = __ffs(m) - 1;
    int base = 0;
    if (b >= 0 && lane == leader) base = atomicAdd(&cnt[b], __popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (b >= 0) perm[base + __popc(m & ((1u << lane) - 1u))] = i;
  }
}

// precision mode 2 (device reference): every environment goes to the fp64 path
__global__ void slam_fill_list_kernel(int N, int* list, int* cnt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) list[i] = i;
  if (i == 0) cnt[0] = N;
}

// reset: one warp per environment
__global__ void slam_reset_kernel(Layout ly, Params pr, float* state, const float* init_pose, int* perm, int* keys) {
  const int env = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (env >= ly.N) return;
  if (lane == 0) { perm[env] = env; keys[env] = 0; }
  float* rec = state + (size_t)env * ly.rec;
  int* reci = reinterpret_cast<int*>(rec);
  for (int i = lane; i < ly.o_lam + 8; i += 32) rec[i] = 0.f;
  __syncwarp();
  for (int k = lane; k < ly.W; k += 32) reci[ly.o_lct + k] = -1;
  if (lane < 3) {
    const float a = init_pose ? init_pose[(size_t)lane * ly.N + env] : 0.f;
    rec[ly.o_a + lane] = a;
    rec[ly.o_vbar + lane] = a;
    rec[ly.o_lam + (lane * (lane + 1) / 2) + lane] = pr.om_prior[lane];
  }
}

// NEXT-2: per-environment episode reset (episodes end after 2048 steps or on collision).
// One warp per environment; only environments with mask != 0 are touched.
__global__ void slam_reset_envs_kernel(Layout ly, Params pr, float* state, int c, const int32_t* mask, const float* init_pose) {
  const int env = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (env >= ly.N || mask[env] == 0) return;
  float* rec = state + (size_t)env * ly.rec;
  int* reci = reinterpret_cast<int*>(rec);
  for (int i = lane; i < ly.o_a; i += 32) rec[i] = 0.f;                 // status, support / active / unary masks
  for (int i = ly.o_vbar + lane; i < ly.o_lam + 8; i += 32) rec[i] = 0.f;
  for (int i = lane; i < ly.W * ly.nw; i += 32) rec[ly.o_rbm + i] = 0.f;   // the new anchor slot observes nothing
  for (int k = lane; k < ly.W; k += 32) reci[ly.o_lct + k] = -1;
  __syncwarp();
  if (lane == 0) reci[ly.o_k0] = c - 1;                                  // its window restarts with one pose
  if (lane < 3) {
    const float a = init_pose ? init_pose[(size_t)lane * ly.N + env] : 0.f;
    rec[ly.o_a + lane] = a;
    rec[ly.o_vbar + lane] = a;
    rec[ly.o_lam + (lane * (lane + 1) / 2) + lane] = pr.om_prior[lane];
  }
}

// poses[3][W][N] = a (+) e_k for k < c, else 0
__global__ void slam_poses_kernel(Layout ly, const float* state, const double* state64, int head, int c, float* poses) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= ly.N) return;
  const float* rec = state + (size_t)env * ly.rec;
  const int k0 = reinterpret_cast<const int*>(rec)[ly.o_k0];
  c -= k0;
  head = (head + k0) % ly.W;
  if (reinterpret_cast<const int*>(rec)[ly.o_mode] != 0) {   // the state lives in the fp64 shadow record
    const double* r64 = state64 + (size_t)env * ly.rec;
    const double ax = r64[ly.o_a], ay = r64[ly.o_a + 1], at = r64[ly.o_a + 2], sn = sin(at), cn = cos(at);
    for (int k = 0; k < ly.W; ++k) {
      double x = 0.0, y = 0.0, t = 0.0;
      if (k < c) {
        const int r = ring_of(k, head, ly.W);
        const double ex = k ? r64[ly.o_e + 3 * r] : 0.0, ey = k ? r64[ly.o_e + 3 * r + 1] : 0.0, et = k ? r64[ly.o_e + 3 * r + 2] : 0.0;
        x = ax + cn * ex - sn * ey; y = ay + sn * ex + cn * ey; t = slamr::wrapr(at + et);
      }
      poses[((size_t)0 * ly.W + k) * ly.N + env] = (float)x;
      poses[((size_t)1 * ly.W + k) * ly.N + env] = (float)y;
      poses[((size_t)2 * ly.W + k) * ly.N + env] = (float)t;
    }
    return;
  }
  const float ax = rec[ly.o_a], ay = rec[ly.o_a + 1], at = rec[ly.o_a + 2];
  float sn, cn;
  sincos_pi(at, &sn, &cn);
  for (int k = 0; k < ly.W; ++k) {
    float x = 0.f, y = 0.f, t = 0.f;
    if (k < c) {
      const int r = ring_of(k, head, ly.W);
      const float ex = k ? rec[ly.o_e + 3 * r] : 0.f, ey = k ? rec[ly.o_e + 3 * r + 1] : 0.f, et = k ? rec[ly.o_e + 3 * r + 2] : 0.f;
      x = ax + cn * ex - sn * ey; y = ay + sn * ex + cn * ey; t = wrapf(at + et);
    }
    poses[((size_t)0 * ly.W + k) * ly.N + env] = x;
    poses[((size_t)1 * ly.W + k) * ly.N + env] = y;
    poses[((size_t)2 * ly.W + k) * ly.N + env] = t;
  }
}

__global__ void slam_landmarks_kernel(Layout ly, const float* state, const double* state64, float* lm, uint32_t* active) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= ly.N) return;
  const float* rec = state + (size_t)env * ly.rec;
  const double* r64 = state64 + (size_t)env * ly.rec;
  const uint32_t* recu = reinterpret_cast<const uint32_t*>(rec);
  const bool m64 = recu[ly.o_mode] != 0;
  for (int q = 0; q < ly.nw; ++q) active[(size_t)q * ly.N + env] = recu[ly.o_act + q];
  for (int l = 0; l < ly.L; ++l) {
    const bool act = (recu[ly.o_act + (l >> 5)] >> (l & 31)) & 1u;
    const float mx = m64 ? (float)r64[ly.o_m + 2 * l] : rec[ly.o_m + 2 * l], my = m64 ? (float)r64[ly.o_m + 2 * l + 1] : rec[ly.o_m + 2 * l + 1];
    lm[((size_t)0 * ly.L + l) * ly.N + env] = act ? mx : 0.f;  // landmarks are stored in global coordinates
    lm[((size_t)1 * ly.L + l) * ly.N + env] = act ? my : 0.f;
  }
}

__global__ void slam_status_kernel(Layout ly, const float* state, int32_t* status) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env < ly.N) status[env] = reinterpret_cast<const int*>(state + (size_t)env * ly.rec)[ly.o_status];
}

__global__ void slam_copycov_kernel(int N, const float* cache, float* cov, float* logdet, float* dopt) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= N) return;
  if (cov)
    for (int k = 0; k < 9; ++k) cov[(size_t)k * N + env] = cache[(size_t)k * N + env];
  const float ld = cache[(size_t)9 * N + env];
  if (logdet) logdet[env] = ld;
  if (dopt) dopt[env] = expf(ld * (1.0f / 3.0f));
}

// NEXT-4: reward of eqs. (7)-(17), one thread per environment
__global__ void slam_reward_kernel(int N, slam_reward_params p, const float* u, const float* u_prev, const float* dcells,
                                   const float* d_min, const int32_t* collision, float* reward) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= N) return;
  if (collision[env] != 0) { reward[env] = -p.lambda_col; return; }                       // (7)
  const float U = u[env], Up = u_prev[env];
  float cc = fminf(fmaxf((p.u_hi - Up) / p.u_hi, 0.f), 1.f);
  cc *= cc;                                                                               // (11)
  const float drop = Up - U;
  const float iota = fminf(fmaxf(fmaxf(drop, 0.f) / p.kappa, 0.f), 1.f);                  // (12)
  const float I = cc + (1.f - cc) * iota;                                                 // (10)
  const float r_explore = p.lambda_explore * dcells[env] * I;                             // (8)
  const float ex = expf(Up);
  const float r_abs = p.lambda_abs * ex * Up;                                             // (13)
  const float r_delta = p.lambda_delta * ex * drop;                                       // (14)
  const float alpha = fminf(fmaxf((d_min[env] - p.d_crash) / (p.d_full - p.d_crash), 0.f), 1.f);  // (15)
  reward[env] = r_explore * alpha - r_abs + (drop > 0.f ? r_delta * alpha : r_delta);     // (16), (17), (7)
}

// Register-resident FP32 FMA microbenchmark (the roofline's FP32 peak has to be MEASURED):
// 16 independent accumulator chains per thread, no memory traffic inside the loop; 2 flop per FMA.
__global__ void __launch_bounds__(256) slam_fma_probe_kernel(long long iters, float a, float b, float* sink) {
  float acc[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (long long i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int k = 0; k < 16; ++k) acc[k] = fmaf(acc[k], a, b);
  }
  float t = 0.f;
#pragma unroll
  for (int k = 0; k < 16; ++k) t += acc[k];
  if (t == 123.456f) sink[0] = t;   // (never true for the arguments used: keeps the chains alive)
}

// ------------------------------------------------------------------ host object
struct slam_ctx {
  Layout ly;
  Params pr;
  cudaStream_t stream;
  int device;                 // the CUDA device the context was created on (every call makes it current)
  float* state;
  float* cov_cache;
  unsigned long long* stats;  // [8] device counters: max / sum / count of envelope words, ...
  int *perm, *keys;           // [N] cost order of the environments and the keys it is sorted by
  // fp64 path (slam_ref64.cuh): shadow records, the list of environments it has to process, launch shape
  double* state64;
  int *fb_list, *fb_cnt;
  double* hglob;
  int precision;              // 0: fp32 only, 1: fp32 with fp64 fallback on ill-conditioned windows, 2: fp64 everywhere
  bool precision_auto;        // the default rule decides (landmarks or unary factors -> 1, else 0)
  float ratio_hi, ratio_lo;
  int min_vis;                // landmarks the newest pose must see before an fp64 environment goes back to fp32
  int box_vis;                // ... and to count as well localised: twice the thresholds (0: never)
  int ref_grid, ref_smem;
  bool order, order_all;      // re-sort after every solve (SLAM_ORDER=0 disables, 1: windows with landmarks only)
  // device staging for slam_step_host
  float *st_odom, *st_lc_meas, *st_rb_meas, *st_cov, *st_logdet, *st_pose;
  int32_t* st_lc_back;
  uint32_t* st_rb_mask;
  int head, count;
  bool cov_valid;
  const float *un_pose, *un_info;   // pending unary factor for the next pushed pose (NEXT-1)
  const int32_t* un_valid;
  long long launches;
  int grid, smem_bytes, ctas_per_sm;
  // optional per-kernel timing of the step launches (slam_kernel_timing): 4 events per step in a ring
  cudaEvent_t* tev;
  int tev_steps, tev_cap;
  char err[256];
};

static int fail(slam_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}
static int check_cuda(slam_ctx* c, const char* what) {
  const cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) return SLAM_OK;
  if (c) snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
  return SLAM_ECUDA;
}
static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }
// Makes the context's device current for the duration of a call (a context created on cuda:1 must not launch on
// whatever device the caller's thread happens to have current).
struct DevGuard {
  int prev;
  bool swapped;
  explicit DevGuard(const slam_ctx* c) : prev(-1), swapped(false) {
    if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) swapped = cudaSetDevice(c->device) == cudaSuccess;
  }
  ~DevGuard() { if (swapped) cudaSetDevice(prev); }
};
static int sm_count() {  // SMs of the current device (148 on B200)
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
    cudaGetLastError();
    sms = 148;
  }
  return sms;
}

static bool sizes_ok(int batch, int window, int landmarks) {
  return batch >= 1 && window >= 2 && window <= SLAM_MAX_WINDOW && landmarks >= 0 && landmarks <= SLAM_MAX_LANDMARKS;
}

// Threads per environment: SLAM_TEAM={32,64,128} overrides.  One warp per environment keeps the most
// environments in flight (the register file holds 15 one-warp teams per SM but only 8 two-warp teams) and
// wins whenever the batch fills the SMs (measured with the pooled shared memory, ms per step, 32 vs 64
// threads: config 2 0.39 / 0.61, config 3 2.36 / 2.70, config 4 3.44 / 3.51); a small batch (config 1:
// 750 environments = 5 per SM) is latency bound and prefers two warps per environment (0.135 / 0.108).
static int pick_team(int W, int L, int batch) {
  const char* e = getenv("SLAM_TEAM");
  if (e) { const int t = atoi(e); if (t == 32 || t == 64 || t == 128) return t; }
  const int n = 3 * W + 2 * L;
  if (n >= 48 && batch < sm_count() * 8) return 64;
  return 32;
}
static int max_teams(int team) {  // threads per CTA: register file (launch bounds), 15 named barriers, 16 table slots
  int maxt = team == 128 ? 7 : SLAM_MAXTHREADS / team;   // (32 threads: 16 teams = the whole register file)
  if (maxt > (team == 32 ? 16 : 15)) maxt = team == 32 ? 16 : 15;
  const char* e = getenv("SLAM_MAX_WPC");
  if (e && atoi(e) >= 1 && atoi(e) < maxt) maxt = atoi(e);
  return maxt;
}
// Teams per CTA and words of the CTA pool.  More teams = more environments in flight but a smaller pool
// (each team has a fixed part); the expected number in flight is min(teams, pool / typical need) with the
// typical need a fraction of the dense size.  Measured (ms per step by teams per SM): config 3: 14 2.19,
// 15 2.25, 16 2.13; config 4: 12 3.20, 13 3.23, 14 3.18, 15 3.37, 16 3.20 (rows in pairs: 14 2.95, 16 2.91)
// -- rather a full pool with some
// teams waiting than idle shared memory, hence fractions below the measured mean envelopes (0.5 / 0.33).
// SLAM_TYPICAL_FRAC overrides; SLAM_POOL_FRAC (0..1] shrinks the pool (tests: forces waiting).
static const int SMEM_BUDGET = 227 * 1024 - 512;  // dynamic shared memory per CTA (static tables: < 512 B)
static int pick_launch(int W, int L, int team, int pairs, int* pool_words) {
  const Layout d = make_layout(1, W, L, 0, 1);
  double tf = L > 0 ? 0.4 : 0.24;
  { const char* e = getenv("SLAM_TYPICAL_FRAC"); if (e && atof(e) > 0.0 && atof(e) <= 1.0) tf = atof(e); }
  const double typical = tf * d.dense;
  int best = 0, best_pool = 0;
  double best_est = 0.0;
  // ctas = 2: two smaller CTAs per SM, each with its own pool, when the estimate loses no environment in
  // flight: the lock-step rounds of the two CTAs drift apart, so one CTA's work fills the tail of the
  // other's round (measured, ms per step, one / two CTAs: config 1 0.107 / 0.102, config 2 0.393 / 0.384,
  // config 3 2.076 / 2.043; config 4, whose windows need half a pool of 8 teams and more, 2.845 / 3.004:
  // the estimate keeps it on one CTA).  SLAM_SPLIT_CTA=0 disables.
  const char* sp = getenv("SLAM_SPLIT_CTA");
  const int max_ctas = ((sp && sp[0] == '0') || (pairs && !(sp && sp[0] == '2'))) ? 1 : 2;   // (rows in pairs = shared memory binds: one pool; SLAM_SPLIT_CTA=2 tries two anyway)
  for (int ctas = 1; ctas <= max_ctas; ++ctas) {
    const int budget = ctas == 1 ? SMEM_BUDGET : (228 * 1024 / 2 - 1024 - 512);
    for (int wpc = 1; wpc * ctas <= max_teams(team); ++wpc) {
      const int pool = (budget / 4 - wpc * d.team_words) & ~3;
      if (pool < d.dense) break;
      if (wpc > 4 && (wpc & 1)) continue;  // even team counts load the four sub-partitions evenly (measured: 15 teams slower than 14 and 16)
      const double fit = pool / typical;
      double est = ctas * (fit < wpc ? fit : wpc);
      if (ctas == 2) est += 0.25;  // at equal expected occupancy prefer two CTAs
      if (est > best_est + 1e-9) { best_est = est; best = wpc; best_pool = pool; }
    }
  }
  const char* e = getenv("SLAM_POOL_FRAC");
  if (best && e) { const double f = atof(e); if (f > 0.0 && f <= 1.0) { best_pool = (int)(f * best_pool) & ~3; if (best_pool < d.dense) best_pool = d.dense; } }
  *pool_words = best_pool;
  return best;  // 0 if one environment does not fit
}
typedef void (*step_fn)(Layout, Params, float*, int, int, int, int, StepIO, unsigned long long*, const int*, int*, int*, int*);
template <bool PAIRS, bool LM>
[[maybe_unused]] static step_fn kernel_pick(int team) {
  return team == 128 ? slam_step_kernel<128, PAIRS, LM> : (team == 64 ? slam_step_kernel<64, PAIRS, LM> : slam_step_kernel<32, PAIRS, LM>);
}
// One instantiation per (team size, envelope rows in pairs, window has landmarks): the pose-only kernels
// carry no code for cached landmark columns, the fours kernels none for split dot products.
static step_fn kernel_of(int team, int pairs, int landmarks) {
#ifdef SLAM_DEV_SINGLE   // developer build (compiles in a fifth of the time): only the kernels of BASELINE configs 3 and 4
  return landmarks ? slam_step_kernel<32, true, true> : slam_step_kernel<32, true, false>;
#else
  if (pairs) return landmarks ? kernel_pick<true, true>(team) : kernel_pick<true, false>(team);
  return landmarks ? kernel_pick<false, true>(team) : kernel_pick<false, false>(team);
#endif
}
// Envelope rows in pairs instead of fours: 12-18 % fewer shared-memory words per environment, ~5 % more
// instructions.  Pays where the pool bounds the environments in flight: at a third of the dense size per
// environment for pose-only windows (measured, ms per step, fours / pairs: config 4 3.48 / 3.09, config 2 0.373 /
// 0.417), at half of it for windows with landmarks, whose envelope is denser (config 3 while the robots are among
// the landmarks: 2.46 / 2.33, pool waits halved; over the whole 300 steps, whose late windows are nearly empty,
// 1.72 / 1.76 -- the dear phase decides).  SLAM_PAIRS=0/1 overrides.
static int pick_pairs(int W, int L, int team) {
  const char* e = getenv("SLAM_PAIRS");
  if (e && (e[0] == '0' || e[0] == '1')) return e[0] == '1';
  const Layout d = make_layout(1, W, L, 0, 1);
  return team == 32 && 16.0 * (d.team_words + (L > 0 ? 0.5 : 0.3) * d.dense) > SMEM_BUDGET / 4;
}

// The ONE place that decides the launch shape of the step kernel for given sizes (slam_workspace_bytes and
// slam_create both go through it): threads per environment, envelope grouping, teams per CTA, pool words.
static bool pick_layout(int batch, int window, int landmarks, Layout* out) {
  const int team = pick_team(window, landmarks, batch);
  const int pairs = pick_pairs(window, landmarks, team);
  int pool = 0;
  const int wpc = pick_launch(window, landmarks, team, pairs, &pool);
  if (wpc < 1) return false;
  *out = make_layout(batch, window, landmarks, pool, wpc);
  out->team = team;
  out->pairs = pairs;
  return true;
}

// fp64 path: dynamic shared memory of one CTA (everything but H, plus H when it fits) and the global scratch
// for H when it does not (one packed triangle per resident CTA; grid = 2 CTAs per SM then)
static const int REF_MAX_GRID_GLOBAL = 2 * 160;
static size_t ref_small_bytes(const Layout& ly) { return slamr::ref_smem_doubles(ly) * 8 + slamr::ref_smem_ints(ly) * 4 + 32; }
static bool ref_h_in_smem(const Layout& ly) { return ref_small_bytes(ly) + slamr::ref_tri(ly) * 8 <= (size_t)SMEM_BUDGET; }
static size_t ref_hglob_bytes(const Layout& ly) { return ref_h_in_smem(ly) ? 0 : (size_t)REF_MAX_GRID_GLOBAL * slamr::ref_tri(ly) * 8; }
struct WsPlan { size_t stats, perm, keys, state, cache, odom, lcb, lcm, rbk, rbm, cov, ld, pose, fbl, fbc, s64, hg, total; };
static WsPlan plan(const Layout& ly) {
  WsPlan p;
  size_t o = 0;
  const size_t N = (size_t)ly.N;
  p.stats = o; o = al256(o + 256);
  p.perm = o; o = al256(o + N * 4);
  p.keys = o; o = al256(o + N * 4);
  p.state = o; o = al256(o + N * ly.rec * 4);
  p.cache = o; o = al256(o + N * 10 * 4);
  p.odom = o; o = al256(o + N * 3 * 4);
  p.lcb = o; o = al256(o + N * 4);
  p.lcm = o; o = al256(o + N * 3 * 4);
  p.rbk = o; o = al256(o + N * (size_t)(ly.nw ? ly.nw : 1) * 4);
  p.rbm = o; o = al256(o + N * (size_t)(ly.L ? 2 * ly.L : 1) * 4);
  p.cov = o; o = al256(o + N * 9 * 4);
  p.ld = o; o = al256(o + N * 4);
  p.pose = o; o = al256(o + N * 3 * 4);
  p.fbl = o; o = al256(o + N * 4);
  p.fbc = o; o = al256(o + 64);
  p.s64 = o; o = al256(o + N * ly.rec * 8);
  p.hg = o; o = al256(o + ref_hglob_bytes(ly));
  p.total = o;
  return p;
}

extern "C" {

void slam_default_config(slam_config* cfg) {
  if (!cfg) return;
  const float p[3] = {0.01f, 0.01f, 0.005f}, o[3] = {0.05f, 0.05f, 0.02f}, l[3] = {0.10f, 0.10f, 0.03f};
  for (int k = 0; k < 3; ++k) { cfg->prior_sigma[k] = p[k]; cfg->odo_sigma[k] = o[k]; cfg->lc_sigma[k] = l[k]; }
  cfg->rb_sigma[0] = 0.05f; cfg->rb_sigma[1] = 0.01f;
}

size_t slam_workspace_bytes(int batch, int window, int landmarks) {
  if (!sizes_ok(batch, window, landmarks)) return 0;
  Layout ly;
  if (!pick_layout(batch, window, landmarks, &ly)) return 0;
  return plan(ly).total;
}

int slam_create(slam_ctx** out, int batch, int window, int landmarks, const slam_config* cfg, void* workspace,
                size_t workspace_bytes, void* cuda_stream) {
  if (!out) return SLAM_EINVAL;
  *out = nullptr;
  if (!sizes_ok(batch, window, landmarks) || !workspace || ((uintptr_t)workspace & 255)) return SLAM_EINVAL;
  Layout ly0;
  if (!pick_layout(batch, window, landmarks, &ly0)) return SLAM_EINVAL;
  const int team = ly0.team, wpc = ly0.wpc;
  slam_config dc;
  slam_default_config(&dc);
  if (!cfg) cfg = &dc;
  for (int k = 0; k < 3; ++k)
    if (!(cfg->prior_sigma[k] > 0.f) || !(cfg->odo_sigma[k] > 0.f) || !(cfg->lc_sigma[k] > 0.f)) return SLAM_EINVAL;
  if (!(cfg->rb_sigma[0] > 0.f) || !(cfg->rb_sigma[1] > 0.f)) return SLAM_EINVAL;
  slam_ctx* c = new (std::nothrow) slam_ctx();
  if (!c) return SLAM_ENOMEM;
  c->ly = ly0;
  if (cudaGetDevice(&c->device) != cudaSuccess) { cudaGetLastError(); delete c; return SLAM_ECUDA; }
  { const char* e = getenv("SLAM_LOCK"); if (e) c->ly.lock = atoi(e); }
  { const char* e = getenv("SLAM_LCACHE"); if (e) c->ly.lcache = atoi(e); }
  { const char* e = getenv("SLAM_DYNQ"); c->ly.dynq = e ? atoi(e) : 1; }
  // Bytes of the next round's records the step kernel prefetches into L2.  OFF by default: measured -0.4 % on the
  // step kernel for +45 % DRAM traffic and no drop of the long-scoreboard share.
  // SLAM_PREFETCH=1: everything up to the prior mean and gradient plus the packed Lambda of a typical support (a
  // third of the state); SLAM_PREFETCH=<bytes>: that many.
  {
    const int s_typ = c->ly.n / 3 + 6;
    long long b = 4ll * (c->ly.o_lam + s_typ * (s_typ + 1) / 2);
    if (b > 4ll * c->ly.rec) b = 4ll * c->ly.rec;
    const char* e = getenv("SLAM_PREFETCH");
    const int v = e ? atoi(e) : 0;
    c->ly.pf_bytes = v <= 0 ? 0 : (v == 1 ? (int)(b & ~15ll) : (int)((v < 4ll * c->ly.rec ? v : 4ll * c->ly.rec) & ~15ll));
  }
  const WsPlan p = plan(c->ly);
  if (workspace_bytes < p.total) { delete c; return SLAM_EINVAL; }
  for (int k = 0; k < 3; ++k) {
    c->pr.om_prior[k] = 1.0f / (cfg->prior_sigma[k] * cfg->prior_sigma[k]);
    c->pr.om_odo[k] = 1.0f / (cfg->odo_sigma[k] * cfg->odo_sigma[k]);
    c->pr.om_lc[k] = 1.0f / (cfg->lc_sigma[k] * cfg->lc_sigma[k]);
  }
  c->pr.om_rb[0] = 1.0f / (cfg->rb_sigma[0] * cfg->rb_sigma[0]);
  c->pr.om_rb[1] = 1.0f / (cfg->rb_sigma[1] * cfg->rb_sigma[1]);
  c->stream = (cudaStream_t)cuda_stream;
  char* base = (char*)workspace;
  c->stats = (unsigned long long*)(base + p.stats);
  c->perm = (int*)(base + p.perm);
  c->keys = (int*)(base + p.keys);
  { const char* e = getenv("SLAM_ORDER"); c->order = !(e && e[0] == '0'); c->order_all = !(e && e[0] == '1'); }
  c->state = (float*)(base + p.state);
  c->cov_cache = (float*)(base + p.cache);
  c->st_odom = (float*)(base + p.odom);
  c->st_lc_back = (int32_t*)(base + p.lcb);
  c->st_lc_meas = (float*)(base + p.lcm);
  c->st_rb_mask = (uint32_t*)(base + p.rbk);
  c->st_rb_meas = (float*)(base + p.rbm);
  c->st_cov = (float*)(base + p.cov);
  c->st_logdet = (float*)(base + p.ld);
  c->st_pose = (float*)(base + p.pose);
  c->launches = 0;
  c->tev = nullptr; c->tev_steps = 0; c->tev_cap = 0;
  c->err[0] = 0;
  c->un_pose = nullptr; c->un_info = nullptr; c->un_valid = nullptr;
  c->fb_list = (int*)(base + p.fbl);
  c->fb_cnt = (int*)(base + p.fbc);
  c->state64 = (double*)(base + p.s64);
  c->hglob = ref_h_in_smem(c->ly) ? nullptr : (double*)(base + p.hg);
  // Precision.  Pose-only windows without absolute measurements keep the anchor out of
  // every factor: fp32 holds the tolerances with a wide margin and the watch is off.  Landmarks (global, so every
  // range-bearing factor touches the anchor) and unary factors switch it on: slam_set_precision overrides.
  c->precision_auto = true;
  c->precision = landmarks > 0 ? 1 : 0;
  c->ratio_hi = 300.f; c->ratio_lo = 150.f;
  c->min_vis = 3;
  c->box_vis = 9;
  { const char* e = getenv("SLAM_BOX_VIS"); if (e) c->box_vis = atoi(e); }
  { const char* e = getenv("SLAM_MIN_VIS"); if (e) c->min_vis = atoi(e); }
  { const char* e = getenv("SLAM_RATIO_HI"); if (e && atof(e) > 0) c->ratio_hi = (float)atof(e); e = getenv("SLAM_RATIO_LO"); if (e && atof(e) > 0) c->ratio_lo = (float)atof(e); }
  { const char* e = getenv("SLAM_PRECISION"); if (e && e[0] >= '0' && e[0] <= '2') { c->precision = e[0] - '0'; c->precision_auto = false; } }
  c->ref_smem = (int)(ref_small_bytes(c->ly) + (c->hglob ? 0 : slamr::ref_tri(c->ly) * 8));
  if (cudaFuncSetAttribute(slamr::slam_ref64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET) != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return SLAM_ECUDA;
  }
  c->smem_bytes = (c->ly.team_words * wpc + c->ly.pool) * 4;
  if (cudaFuncSetAttribute(kernel_of(team, c->ly.pairs, c->ly.L), cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET) != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return SLAM_ECUDA;
  }
  int dev = 0, sms = 0, occ = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel_of(team, c->ly.pairs, c->ly.L), wpc * team, c->smem_bytes);
  if (occ < 1 || sms < 1) { cudaGetLastError(); delete c; return SLAM_ECUDA; }
  c->ctas_per_sm = occ;
  const int need = (batch + wpc - 1) / wpc;
  c->grid = need < sms * occ ? need : sms * occ;
  {
    int rocc = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&rocc, slamr::slam_ref64_kernel, slamr::NT, c->ref_smem);
    if (rocc < 1) { cudaGetLastError(); delete c; return SLAM_ECUDA; }
    long long g = (long long)sms * rocc;
    if (c->hglob && g > REF_MAX_GRID_GLOBAL) g = REF_MAX_GRID_GLOBAL;
    c->ref_grid = (int)(g < batch ? g : batch);
  }
  *out = c;
  const int rc = slam_reset(c, nullptr);
  if (rc != SLAM_OK) { *out = nullptr; slam_destroy(c); }
  return rc;
}

void slam_destroy(slam_ctx* ctx) {
  if (!ctx) return;
  if (ctx->tev) {
    DevGuard dg(ctx);
    for (int i = 0; i < 4 * ctx->tev_cap; ++i) cudaEventDestroy(ctx->tev[i]);
    delete[] ctx->tev;
  }
  delete ctx;
}

int slam_reset(slam_ctx* c, const float* init_pose) {
  if (!c) return SLAM_EINVAL;
  DevGuard dg(c);
  const int threads = 256, blocks = (int)(((size_t)c->ly.N * 32 + threads - 1) / threads);
  cudaMemsetAsync(c->stats, 0, 256, c->stream);
  cudaMemsetAsync(c->fb_cnt, 0, 64, c->stream);
  slam_reset_kernel<<<blocks, threads, 0, c->stream>>>(c->ly, c->pr, c->state, init_pose, c->perm, c->keys);
  c->launches++;
  c->head = 0; c->count = 1; c->cov_valid = false;
  c->un_pose = nullptr; c->un_info = nullptr; c->un_valid = nullptr;   // a pending slam_set_unary belongs to the old episode
  return check_cuda(c, "slam_reset");
}

static int launch_step(slam_ctx* c, int flags, int iters, const StepIO& io) {
  DevGuard dg(c);
  const step_fn fn = kernel_of(c->ly.team, c->ly.pairs, c->ly.L);
  cudaEvent_t* tv = (c->tev && c->tev_steps < c->tev_cap) ? c->tev + 4 * c->tev_steps : nullptr;
  if (tv) cudaEventRecord(tv[0], c->stream);
  if (c->precision == 2) {   // device reference: every environment through the fp64 path
    const int threads = 256, blocks = (c->ly.N + threads - 1) / threads;
    slam_fill_list_kernel<<<blocks, threads, 0, c->stream>>>(c->ly.N, c->fb_list, c->fb_cnt);
    c->launches++;
  } else {
    Layout ly = c->ly;
    ly.ratio_hi = c->precision == 1 ? c->ratio_hi : 0.f;
    ly.box_vis = c->box_vis;
    fn<<<c->grid, c->ly.wpc * c->ly.team, c->smem_bytes, c->stream>>>(ly, c->pr, c->state, c->head, c->count, flags, iters, io,
                                                                        c->stats, c->perm, c->keys,
                                                                        c->precision == 1 ? c->fb_list : nullptr, c->fb_cnt);
    c->launches++;
  }
  if (tv) cudaEventRecord(tv[1], c->stream);
  if (c->precision >= 1) {   // the environments the fp32 kernel queued: fp64 records, and the windows it refused to commit
    slamr::RefArgs ra = {c->state, c->state64, c->head, c->count, flags, iters, c->fb_list, c->fb_cnt, c->stats, c->hglob,
                         (double)c->ratio_lo, c->precision == 2 ? 1 : 0, c->min_vis, c->box_vis, c->keys};
#ifdef SLAM_REF_PROFILE
    cudaMemcpyToSymbolAsync(slamr::g_ref_prof, &c->stats, sizeof(c->stats), 0, cudaMemcpyHostToDevice, c->stream);
#endif
    slamr::slam_ref64_kernel<<<c->ref_grid, slamr::NT, c->ref_smem, c->stream>>>(c->ly, c->pr, ra, io);
    c->launches++;
  }
  if (tv) cudaEventRecord(tv[2], c->stream);
  // the solve left fresh cost keys: order the next launches by them (pointless unless every CTA runs
  // several rounds; a small batch is latency bound: one more kernel boundary per step would show).  Landmark
  // windows gain most -- their cost varies most: config 3 2.40 -> 2.31 ms per step under the static deal of
  // round 1; pose-only windows gain since the list is handed out from one queue for the grid (most expensive
  // first = longest-processing-time scheduling): config 4 at N = 16384 3.09 -> 3.04, at 65536 11.7 -> 11.3
  if (c->order && iters > 0 && (c->ly.L > 0 || c->order_all) && (long long)c->ly.N >= 4ll * c->grid * c->ly.wpc) {
    slam_order_kernel<<<1, 1024, 0, c->stream>>>(c->ly.N, c->ly.dense, c->keys, c->perm);
    c->launches++;
  }
  if (tv) { cudaEventRecord(tv[3], c->stream); c->tev_steps++; }
  return check_cuda(c, "slam_step_kernel");
}

static int check_push_args(slam_ctx* c, const float* odom, const int32_t* lc_back, const float* lc_meas,
                           const uint32_t* rb_mask, const float* rb_meas) {
  if (!odom) return fail(c, SLAM_EINVAL, "odom is NULL");
  if (lc_back && !lc_meas) return fail(c, SLAM_EINVAL, "lc_back given without lc_meas");
  if (c->ly.L > 0 && (!rb_mask || !rb_meas)) return fail(c, SLAM_EINVAL, "rb_mask/rb_meas required when landmarks > 0");
  if (c->count >= c->ly.W) return fail(c, SLAM_ESTATE, "push on a full window: marginalize first");
  return SLAM_OK;
}

int slam_push_step(slam_ctx* c, const float* odom, const int32_t* lc_back, const float* lc_meas, const uint32_t* rb_mask,
                   const float* rb_meas) {
  if (!c) return SLAM_EINVAL;
  int rc = check_push_args(c, odom, lc_back, lc_meas, rb_mask, rb_meas);
  if (rc) return rc;
  StepIO io = {odom, lc_back, lc_meas, rb_mask, rb_meas, nullptr, nullptr, nullptr, nullptr, c->cov_cache,
               c->un_pose, c->un_info, c->un_valid};
  c->un_pose = nullptr; c->un_info = nullptr; c->un_valid = nullptr;
  rc = launch_step(c, F_PUSH, 0, io);
  if (rc) return rc;
  c->count++; c->cov_valid = false;
  return SLAM_OK;
}

int slam_set_unary(slam_ctx* c, const float* pose, const float* info, const int32_t* valid) {
  if (!c) return SLAM_EINVAL;
  if ((pose == nullptr) != (info == nullptr)) return fail(c, SLAM_EINVAL, "pose and info must both be given (or both NULL to cancel)");
  c->un_pose = pose; c->un_info = info; c->un_valid = pose ? valid : nullptr;
  if (pose && c->precision_auto && c->precision == 0) c->precision = 1;   // absolute measurements couple the anchor to the window
  return SLAM_OK;
}

int slam_reset_envs(slam_ctx* c, const int32_t* mask, const float* init_pose) {
  if (!c || !mask) return c ? fail(c, SLAM_EINVAL, "mask is NULL") : SLAM_EINVAL;
  DevGuard dg(c);
  const int threads = 256, blocks = (int)(((size_t)c->ly.N * 32 + threads - 1) / threads);
  slam_reset_envs_kernel<<<blocks, threads, 0, c->stream>>>(c->ly, c->pr, c->state, c->count, mask, init_pose);
  c->launches++;
  c->cov_valid = false;
  return check_cuda(c, "slam_reset_envs");
}

int slam_observe_first(slam_ctx* c, const uint32_t* rb_mask, const float* rb_meas) {
  if (!c) return SLAM_EINVAL;
  if (c->ly.L == 0) return SLAM_OK;
  if (!rb_mask || !rb_meas) return fail(c, SLAM_EINVAL, "rb_mask/rb_meas are NULL");
  if (c->count != 1) return fail(c, SLAM_ESTATE, "observe_first is only valid right after reset");
  StepIO io = {nullptr, nullptr, nullptr, rb_mask, rb_meas, nullptr, nullptr, nullptr, nullptr, c->cov_cache};
  c->cov_valid = false;
  return launch_step(c, F_OBS0, 0, io);
}

int slam_solve(slam_ctx* c, int iters) {
  if (!c) return SLAM_EINVAL;
  if (iters < 0) return fail(c, SLAM_EINVAL, "iters < 0");
  if (iters == 0) return SLAM_OK;
  StepIO io = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, c->cov_cache};
  c->cov_valid = false;
  return launch_step(c, 0, iters, io);
}

static int cov_call(slam_ctx* c, float* cov, float* logdet, float* dopt) {
  DevGuard dg(c);
  if (c->cov_valid) {
    const int threads = 256, blocks = (c->ly.N + threads - 1) / threads;
    slam_copycov_kernel<<<blocks, threads, 0, c->stream>>>(c->ly.N, c->cov_cache, cov, logdet, dopt);
    c->launches++;
    return check_cuda(c, "slam_copycov_kernel");
  }
  StepIO io = {nullptr, nullptr, nullptr, nullptr, nullptr, cov, logdet, dopt, nullptr, c->cov_cache};
  const int rc = launch_step(c, F_COV, 0, io);
  if (rc == SLAM_OK) c->cov_valid = true;
  return rc;
}

int slam_marginal_cov(slam_ctx* c, float* cov) {
  if (!c) return SLAM_EINVAL;
  if (!cov) return fail(c, SLAM_EINVAL, "cov is NULL");
  return cov_call(c, cov, nullptr, nullptr);
}

int slam_dopt(slam_ctx* c, float* logdet, float* dopt) {
  if (!c) return SLAM_EINVAL;
  if (!logdet && !dopt) return fail(c, SLAM_EINVAL, "logdet and dopt are both NULL");
  return cov_call(c, nullptr, logdet, dopt);
}

int slam_marginalize_oldest(slam_ctx* c) {
  if (!c) return SLAM_EINVAL;
  if (c->count < 2) return fail(c, SLAM_ESTATE, "marginalize needs count >= 2");
  StepIO io = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, c->cov_cache};
  const int rc = launch_step(c, F_MARG, 0, io);
  if (rc) return rc;
  c->head = (c->head + 1) % c->ly.W;
  c->count--;
  c->cov_valid = false;
  return SLAM_OK;
}

int slam_step(slam_ctx* c, const float* odom, const int32_t* lc_back, const float* lc_meas, const uint32_t* rb_mask,
              const float* rb_meas, int iters, float* cov, float* logdet, float* last_pose) {
  if (!c) return SLAM_EINVAL;
  if (iters < 0) return fail(c, SLAM_EINVAL, "iters < 0");
  int rc = check_push_args(c, odom, lc_back, lc_meas, rb_mask, rb_meas);
  if (rc) return rc;
  const bool marg = (c->count + 1 == c->ly.W);
  StepIO io = {odom, lc_back, lc_meas, rb_mask, rb_meas, cov, logdet, nullptr, last_pose, c->cov_cache,
               c->un_pose, c->un_info, c->un_valid};
  c->un_pose = nullptr; c->un_info = nullptr; c->un_valid = nullptr;
  rc = launch_step(c, F_PUSH | F_COV | (marg ? F_MARG : 0), iters, io);
  if (rc) return rc;
  c->count++;
  c->cov_valid = !marg;
  if (marg) { c->head = (c->head + 1) % c->ly.W; c->count--; }
  return SLAM_OK;
}

int slam_step_host(slam_ctx* c, const float* odom, const int32_t* lc_back, const float* lc_meas, const uint32_t* rb_mask,
                   const float* rb_meas, int iters, float* cov, float* logdet, float* last_pose) {
  if (!c) return SLAM_EINVAL;
  DevGuard dg(c);
  int rc = check_push_args(c, odom, lc_back, lc_meas, rb_mask, rb_meas);
  if (rc) return rc;
  const size_t N = (size_t)c->ly.N;
  // (page-locked host buffers make these copies asynchronous; with pageable memory each one blocks the host
  // until it is done -- the results are the same)
  cudaError_t e = cudaMemcpyAsync(c->st_odom, odom, N * 3 * 4, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess && lc_back) {
    e = cudaMemcpyAsync(c->st_lc_back, lc_back, N * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->st_lc_meas, lc_meas, N * 3 * 4, cudaMemcpyHostToDevice, c->stream);
  }
  if (e == cudaSuccess && c->ly.L > 0) {
    e = cudaMemcpyAsync(c->st_rb_mask, rb_mask, N * c->ly.nw * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->st_rb_meas, rb_meas, N * 2 * c->ly.L * 4, cudaMemcpyHostToDevice, c->stream);
  }
  if (e != cudaSuccess) { cudaGetLastError(); snprintf(c->err, sizeof(c->err), "slam_step_host: input copy: %s", cudaGetErrorString(e)); return SLAM_ECUDA; }
  rc = slam_step(c, c->st_odom, lc_back ? c->st_lc_back : nullptr, lc_back ? c->st_lc_meas : nullptr,
                 c->ly.L > 0 ? c->st_rb_mask : nullptr, c->ly.L > 0 ? c->st_rb_meas : nullptr, iters,
                 cov ? c->st_cov : nullptr, logdet ? c->st_logdet : nullptr, last_pose ? c->st_pose : nullptr);
  if (rc) return rc;
  if (cov) e = cudaMemcpyAsync(cov, c->st_cov, N * 9 * 4, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess && logdet) e = cudaMemcpyAsync(logdet, c->st_logdet, N * 4, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess && last_pose) e = cudaMemcpyAsync(last_pose, c->st_pose, N * 3 * 4, cudaMemcpyDeviceToHost, c->stream);
  if (e != cudaSuccess) { cudaGetLastError(); snprintf(c->err, sizeof(c->err), "slam_step_host: output copy: %s", cudaGetErrorString(e)); return SLAM_ECUDA; }
  return SLAM_OK;
}

int slam_get_poses(slam_ctx* c, float* poses) {
  if (!c || !poses) return SLAM_EINVAL;
  DevGuard dg(c);
  const int threads = 128, blocks = (c->ly.N + threads - 1) / threads;
  slam_poses_kernel<<<blocks, threads, 0, c->stream>>>(c->ly, c->state, c->state64, c->head, c->count, poses);
  c->launches++;
  return check_cuda(c, "slam_poses_kernel");
}

int slam_get_landmarks(slam_ctx* c, float* lm, uint32_t* active) {
  if (!c) return SLAM_EINVAL;
  if (c->ly.L == 0) return SLAM_OK;
  if (!lm || !active) return fail(c, SLAM_EINVAL, "lm/active are NULL");
  DevGuard dg(c);
  const int threads = 128, blocks = (c->ly.N + threads - 1) / threads;
  slam_landmarks_kernel<<<blocks, threads, 0, c->stream>>>(c->ly, c->state, c->state64, lm, active);
  c->launches++;
  return check_cuda(c, "slam_landmarks_kernel");
}

int slam_get_status(slam_ctx* c, int32_t* status) {
  if (!c || !status) return SLAM_EINVAL;
  DevGuard dg(c);
  const int threads = 128, blocks = (c->ly.N + threads - 1) / threads;
  slam_status_kernel<<<blocks, threads, 0, c->stream>>>(c->ly, c->state, status);
  c->launches++;
  return check_cuda(c, "slam_status_kernel");
}

int slam_get_stats(slam_ctx* c, unsigned long long* stats8) {
  if (!c || !stats8) return SLAM_EINVAL;
  DevGuard dg(c);
#ifdef SLAM_REF_PROFILE
  cudaMemcpyAsync(stats8, c->stats + 8, 64, cudaMemcpyDeviceToDevice, c->stream);
#else
  cudaMemcpyAsync(stats8, c->stats, 64, cudaMemcpyDeviceToDevice, c->stream);
#endif
  return check_cuda(c, "slam_get_stats");
}

int slam_reward(slam_ctx* c, const slam_reward_params* p, const float* u, const float* u_prev, const float* dcells,
                const float* d_min, const int32_t* collision, float* reward) {
  if (!c || !p || !u || !u_prev || !dcells || !d_min || !collision || !reward) return c ? fail(c, SLAM_EINVAL, "NULL argument") : SLAM_EINVAL;
  if (!(p->u_hi > 0.f) || !(p->kappa > 0.f) || !(p->d_full > p->d_crash)) return fail(c, SLAM_EINVAL, "u_hi, kappa > 0 and d_full > d_crash required");
  DevGuard dg(c);
  const int threads = 256, blocks = (c->ly.N + threads - 1) / threads;
  slam_reward_kernel<<<blocks, threads, 0, c->stream>>>(c->ly.N, *p, u, u_prev, dcells, d_min, collision, reward);
  c->launches++;
  return check_cuda(c, "slam_reward_kernel");
}

int slam_set_precision(slam_ctx* c, int mode, float ratio_hi, float ratio_lo) {
  if (!c) return SLAM_EINVAL;
  if (mode < -1 || mode > 2) return fail(c, SLAM_EINVAL, "precision mode must be -1 (default rule), 0, 1 or 2");
  if (ratio_hi < 0.f || ratio_lo < 0.f || (ratio_hi > 0.f && ratio_lo > ratio_hi)) return fail(c, SLAM_EINVAL, "need 0 < ratio_lo <= ratio_hi (0 keeps the current value)");
  if (mode == -1) { c->precision_auto = true; c->precision = c->ly.L > 0 ? 1 : 0; }
  else { c->precision_auto = false; c->precision = mode; }
  if (ratio_hi > 0.f) c->ratio_hi = ratio_hi;
  if (ratio_lo > 0.f) c->ratio_lo = ratio_lo;
  if (c->ratio_lo > c->ratio_hi) c->ratio_lo = c->ratio_hi;
  c->cov_valid = false;
  return SLAM_OK;
}

int slam_kernel_timing(slam_ctx* c, int max_steps) {
  if (!c || max_steps < 0 || max_steps > (1 << 16)) return c ? fail(c, SLAM_EINVAL, "max_steps out of range") : SLAM_EINVAL;
  DevGuard dg(c);
  if (c->tev) {
    for (int i = 0; i < 4 * c->tev_cap; ++i) cudaEventDestroy(c->tev[i]);
    delete[] c->tev;
    c->tev = nullptr; c->tev_cap = 0;
  }
  c->tev_steps = 0;
  if (max_steps == 0) return SLAM_OK;
  c->tev = new (std::nothrow) cudaEvent_t[4 * (size_t)max_steps];
  if (!c->tev) return fail(c, SLAM_ENOMEM, "slam_kernel_timing: host allocation failed");
  for (int i = 0; i < 4 * max_steps; ++i)
    if (cudaEventCreate(&c->tev[i]) != cudaSuccess) {
      for (int j = 0; j < i; ++j) cudaEventDestroy(c->tev[j]);
      delete[] c->tev;
      c->tev = nullptr;
      check_cuda(c, "cudaEventCreate");
      return SLAM_ECUDA;
    }
  c->tev_cap = max_steps;
  return SLAM_OK;
}

int slam_kernel_timing_read(slam_ctx* c, double* ms3, int* steps) {
  if (!c || !ms3) return c ? fail(c, SLAM_EINVAL, "ms3 is NULL") : SLAM_EINVAL;
  DevGuard dg(c);
  ms3[0] = ms3[1] = ms3[2] = 0.0;
  if (steps) *steps = c->tev_steps;
  if (c->tev_steps > 0 && cudaEventSynchronize(c->tev[4 * (c->tev_steps - 1) + 3]) != cudaSuccess) return check_cuda(c, "slam_kernel_timing_read");
  for (int i = 0; i < c->tev_steps; ++i)
    for (int k = 0; k < 3; ++k) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, c->tev[4 * i + k], c->tev[4 * i + k + 1]) != cudaSuccess) return check_cuda(c, "cudaEventElapsedTime");
      ms3[k] += (double)ms;
    }
  c->tev_steps = 0;
  return SLAM_OK;
}

int slam_fma_probe(long long iters, float* sink, void* cuda_stream, double* flops) {
  if (iters < 1 || !sink) return SLAM_EINVAL;
  const int blocks = sm_count() * 8, threads = 256;
  slam_fma_probe_kernel<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>(iters, 0.999f, 1e-3f, sink);
  if (flops) *flops = (double)blocks * threads * (double)iters * 64.0 * 2.0;
  return check_cuda(nullptr, "slam_fma_probe_kernel");
}

int slam_count(const slam_ctx* c) { return c ? c->count : -1; }
long long slam_launch_count(const slam_ctx* c) { return c ? c->launches : -1; }
const char* slam_last_error(const slam_ctx* c) { return c ? c->err : "null context"; }

int slam_kernel_info(const slam_ctx* c, int* smem_bytes_per_cta, int* warps_per_cta, int* ctas_per_sm) {
  if (!c) return SLAM_EINVAL;
  if (smem_bytes_per_cta) *smem_bytes_per_cta = c->smem_bytes;
  if (warps_per_cta) *warps_per_cta = c->ly.wpc * c->ly.team / 32;
  if (ctas_per_sm) *ctas_per_sm = c->ctas_per_sm;
  return SLAM_OK;
}

// ------------------------------------------------------------------ allocation-free entry point
// slam_run_static: a whole episode (reset, T fused steps) for callers that cannot allocate device memory (code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Everything the step kernels keep between
// launches -- the environment records, their fp64 shadows, the cost order, the fallback list, the covariance cache
// -- lives in ONE file-scope device array of SLAM_STATIC_MAX_BYTES instead of a caller-allocated workspace.  Every
// GPU that loads the library holds the array until the process exits.  All calls share it: it keeps the last call's
// contents (slam_create's reset clears what must start at zero: records up to the prior, counters, order), and two
// calls that overlap on the GPU (different streams, no dependency) race.
static __device__ __align__(256) unsigned char g_static_ws[SLAM_STATIC_MAX_BYTES];
// In host code `g_static_ws` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current.
static void* g_static_ptr[64];

static int static_fail(char* err, size_t err_len, int code, const char* msg) {
  if (err && err_len) snprintf(err, err_len, "%s", msg);
  return code;
}

int slam_run_static(int batch, int window, int landmarks, int steps, int iters, const slam_config* cfg, const float* odom,
                    const int32_t* lc_back, const float* lc_meas, const uint32_t* rb_mask, const float* rb_meas, float* cov,
                    float* logdet, float* last_pose, void* cuda_stream, char* err, size_t err_len) {
  if (err && err_len) err[0] = 0;
  if (!sizes_ok(batch, window, landmarks) || steps < 0 || iters < 0) return static_fail(err, err_len, SLAM_EINVAL, "slam_run_static: invalid batch / window / landmarks / steps / iters");
  if (!odom && steps > 0) return static_fail(err, err_len, SLAM_EINVAL, "slam_run_static: odom is NULL");
  const size_t need = slam_workspace_bytes(batch, window, landmarks);
  if (need == 0 || need > (size_t)SLAM_STATIC_MAX_BYTES) {
    char msg[200];
    snprintf(msg, sizeof(msg), "slam_run_static: batch=%d window=%d landmarks=%d needs %zu bytes of scratch, the static array holds %zu (SLAM_STATIC_MAX_BYTES): use slam_create with a caller-owned workspace",
             batch, window, landmarks, need, (size_t)SLAM_STATIC_MAX_BYTES);
    return static_fail(err, err_len, SLAM_ENOMEM, msg);
  }
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return static_fail(err, err_len, SLAM_ECUDA, "slam_run_static: no current CUDA device"); }
  if (!g_static_ptr[dev]) {   // set-up, once per device, with that device current
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_ws);
    if (e != cudaSuccess || !ptr) { cudaGetLastError(); return static_fail(err, err_len, SLAM_ECUDA, cudaGetErrorString(e)); }
    g_static_ptr[dev] = ptr;
  }
  slam_ctx* c = nullptr;   // (a ~1 KB host object; no CUDA allocation of any kind on this path)
  int rc = slam_create(&c, batch, window, landmarks, cfg, g_static_ptr[dev], (size_t)SLAM_STATIC_MAX_BYTES, cuda_stream);
  if (rc != SLAM_OK) return static_fail(err, err_len, rc, "slam_run_static: slam_create on the static array failed");
  const size_t N = (size_t)batch, nw = (size_t)c->ly.nw, L = (size_t)landmarks;
  if (landmarks > 0) rc = slam_observe_first(c, rb_mask, rb_meas);
  for (int t = 1; rc == SLAM_OK && t <= steps; ++t) {
    const size_t q = (size_t)(t - 1);
    rc = slam_step(c, odom + q * 3 * N, lc_back ? lc_back + q * N : nullptr, lc_back ? lc_meas + q * 3 * N : nullptr,
                   landmarks > 0 ? rb_mask + (size_t)t * nw * N : nullptr, landmarks > 0 ? rb_meas + (size_t)t * 2 * L * N : nullptr, iters,
                   cov ? cov + q * 9 * N : nullptr, logdet ? logdet + q * N : nullptr, last_pose ? last_pose + q * 3 * N : nullptr);
  }
  if (rc != SLAM_OK) static_fail(err, err_len, rc, c->err);
  slam_destroy(c);
  return rc;
}

}  // extern "C"
