// NEXT-3: batched correlative scan matcher and log-odds occupancy-grid update (PAPER.md:146, 150-152,
// 165; readings R28-R34 of DESIGN.md).  One CTA per environment.
//
// Precision: the cell an end point falls into is an INTEGER decision, so it is taken in fp64 on both
// sides (the oracle is fp64); grid values, the logistic and the score sums are fp32.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#include "../../include/slam.h"

namespace {

constexpr int kThreads = 128;
constexpr double kPi = 3.14159265358979323846;

__device__ __forceinline__ double ray_angle(int i, int R) { return -0.5 * kPi + i * (kPi / (R - 1)); }

// scores of all candidates of one environment; best and second best
__global__ void __launch_bounds__(kThreads) scan_match_kernel(slam_scan_params p, int N, const float* __restrict__ grid,
                                                               const float* __restrict__ pose_pred,
                                                               const float* __restrict__ ranges, float* pose_meas,
                                                               float* score, float* second, int occ_in_smem) {
  extern __shared__ double sm_d[];
  const int env = blockIdx.x, tid = threadIdx.x;
  const int R = p.R, G = p.G, nt = 2 * p.ht + 1, ny = 2 * p.hy + 1, nx = 2 * p.hx + 1;
  double* cs = sm_d;                                   // [nt][R][2] cos/sin of theta + dtheta + phi_i, times range
  float* rr = reinterpret_cast<float*>(cs + (size_t)nt * R * 2);   // [R] range, <0 = invalid
  float* occ = rr + ((R + 3) & ~3);                                  // [G][G] occupancy probabilities (if they fit)
  __shared__ float best_s[kThreads], sec_s[kThreads];
  __shared__ int best_i[kThreads];
  __shared__ int nvalid_s;
  const double px = (double)pose_pred[env], py = (double)pose_pred[(size_t)N + env], pth = (double)pose_pred[2 * (size_t)N + env];
  if (tid == 0) nvalid_s = 0;
  __syncthreads();
  for (int i = tid; i < R; i += kThreads) {
    const float r = ranges[(size_t)i * N + env];
    const bool ok = r >= p.r_min && r <= p.r_max;
    rr[i] = ok ? r : -1.f;
    if (ok) atomicAdd(&nvalid_s, 1);
  }
  __syncthreads();
  for (int q = tid; q < nt * R; q += kThreads) {
    const int it = q / R, i = q - it * R;
    const double a = pth + (double)((it - p.ht) * p.sth) + ray_angle(i, R);
    const double r = (double)rr[i];
    cs[2 * q] = r * cos(a);
    cs[2 * q + 1] = r * sin(a);
  }
  __syncthreads();
  const int nvalid = nvalid_s;
  const float* g = grid + (size_t)env * G * G;
  if (occ_in_smem) {  // logistic once per cell instead of once per (candidate, ray): 441 x 128 gathers vs G*G cells
    for (int q = tid; q < G * G; q += kThreads) occ[q] = 1.f / (1.f + __expf(-g[q]));
    __syncthreads();
  }
  const double o = -0.5 * G * (double)p.res, ires = 1.0 / (double)p.res;
  float b1 = -1.f, b2 = -1.f;
  int bi = 0x7fffffff;
  const int C = nt * ny * nx;
  for (int c = tid; c < C; c += kThreads) {
    const int it = c / (ny * nx), rem = c - it * ny * nx, iy = rem / nx, ix = rem - iy * nx;
    const double cx = px + (double)((ix - p.hx) * p.sxy), cy = py + (double)((iy - p.hy) * p.sxy);
    const double* t = cs + (size_t)it * R * 2;
    float sum = 0.f;
    for (int i = 0; i < R; ++i) {
      if (rr[i] < 0.f) continue;
      // R28/R31: the same expression as the oracle, in fp64: floor((x - o) / res)
      const int jx = (int)floor((cx + t[2 * i] - o) * ires), jy = (int)floor((cy + t[2 * i + 1] - o) * ires);
      if (jx >= 0 && jx < G && jy >= 0 && jy < G)
        sum += occ_in_smem ? occ[jy * G + jx] : 1.f / (1.f + __expf(-__ldg(g + (size_t)jy * G + jx)));
    }
    const float s = nvalid ? sum / (float)nvalid : 0.f;
    if (s > b1) { b2 = b1; b1 = s; bi = c; }      // candidates visited in increasing index: ties keep the lowest
    else if (s > b2) b2 = s;
  }
  best_s[tid] = b1; sec_s[tid] = b2; best_i[tid] = bi;
  __syncthreads();
  if (tid == 0) {
    float g1 = -1.f;
    int gi = 0x7fffffff;
    for (int k = 0; k < kThreads; ++k)
      if (best_s[k] > g1 || (best_s[k] == g1 && best_i[k] < gi)) { g1 = best_s[k]; gi = best_i[k]; }
    float g2 = -1.f;
    for (int k = 0; k < kThreads; ++k) {
      const float v = (best_i[k] == gi) ? sec_s[k] : best_s[k];
      if (v > g2) g2 = v;
    }
    if (g2 < 0.f) g2 = 0.f;
    const int it = gi / (ny * nx), rem = gi - it * ny * nx, iy = rem / nx, ix = rem - iy * nx;
    pose_meas[env] = (float)(px + (double)((ix - p.hx) * p.sxy));
    pose_meas[(size_t)N + env] = (float)(py + (double)((iy - p.hy) * p.sxy));
    pose_meas[2 * (size_t)N + env] = (float)(pth + (double)((it - p.ht) * p.sth));
    score[env] = g1;
    second[env] = g2;
  }
}

// Lattice variant: the xy step of the candidates is a whole number `m` of cells (sxy == m * res, true for every
// configuration used).  The cell of a ray's end point then moves by exactly m cells per xy step, so it is decided
// ONCE per (theta candidate, ray) with the oracle's fp64 expression and the (2hx+1)(2hy+1) xy candidates are integer
// index shifts of it: no fp64 and no floor in the inner loop (49 x fewer at hx = hy = 3).  An end point within
// `margin` cells of a cell edge could fall either way under the rounding of the candidate offset
// ((ix - hx) * sxy is rounded to float first, as in the general kernel): those rays (a few per million) keep the
// exact expression per candidate, so every integer decision is the one the general kernel takes.
// One thread per candidate, lanes along ix: the gathers of a warp are runs of consecutive cells.
// Block size = the candidate count rounded up to whole warps (at most kLatMax): one candidate per thread.
constexpr int kLatMax = 512;
__global__ void __launch_bounds__(kLatMax) scan_match_lattice_kernel(slam_scan_params p, int N, int m, const float* __restrict__ grid,
                                                                          const float* __restrict__ pose_pred,
                                                                          const float* __restrict__ ranges, float* pose_meas,
                                                                          float* score, float* second, int occ_in_smem) {
  extern __shared__ double sm_d[];
  const int env = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int R = p.R, G = p.G, nt = 2 * p.ht + 1, ny = 2 * p.hy + 1, nx = 2 * p.hx + 1;
  double* cs = sm_d;                                            // [nt][R][2] range * cos/sin(theta + dtheta + phi_i)
  int* cell = reinterpret_cast<int*>(cs + (size_t)nt * R * 2);  // [nt][R] base cell: jx + 32768 | (jy + 32768) << 16; 0: edge ray
  float* rr = reinterpret_cast<float*>(cell + (size_t)nt * R);  // [R] range, < 0 = invalid
  float* occ = rr + ((R + 3) & ~3);                              // [G][G] occupancy probabilities (occ_in_smem)
  const int kLatThreads = blockDim.x;
  __shared__ float w_b1[kLatMax / 32], w_b2[kLatMax / 32];
  __shared__ int w_bi[kLatMax / 32];
  __shared__ int nvalid_s;
  const double px = (double)pose_pred[env], py = (double)pose_pred[(size_t)N + env], pth = (double)pose_pred[2 * (size_t)N + env];
  if (tid == 0) nvalid_s = 0;
  __syncthreads();
  for (int i = tid; i < R; i += kLatThreads) {
    const float r = ranges[(size_t)i * N + env];
    const bool ok = r >= p.r_min && r <= p.r_max;
    rr[i] = ok ? r : -1.f;
    if (ok) atomicAdd(&nvalid_s, 1);
  }
  __syncthreads();
  const double o = -0.5 * G * (double)p.res, ires = 1.0 / (double)p.res;
  const int hmax = p.hx > p.hy ? p.hx : p.hy;
  const double margin = 1e-6 + 2.5e-7 * (double)(hmax * m);     // cells; float rounding of the offset is <= 6e-8 * hmax * m
  for (int q = tid; q < nt * R; q += kLatThreads) {
    const int it = q / R, i = q - it * R;
    const double a = pth + (double)((it - p.ht) * p.sth) + ray_angle(i, R);
    const double r = (double)rr[i];
    const double ex = r * cos(a), ey = r * sin(a);
    cs[2 * q] = ex;
    cs[2 * q + 1] = ey;
    int code = 0x00010001;                                      // invalid ray: cell (-32767, -32767), never inside the grid
    if (r >= 0.0) {
      const double ux = (px + ex - o) * ires, uy = (py + ey - o) * ires;
      const double fx = floor(ux), fy = floor(uy);
      const bool edge = ux - fx < margin || ux - fx > 1.0 - margin || uy - fy < margin || uy - fy > 1.0 - margin;
      const bool far = fabs(fx) > 30000.0 || fabs(fy) > 30000.0;   // (cannot be inside a grid of <= 2048 cells)
      code = edge ? 0 : (far ? 0x00010001 : (((int)fx + 32768) | (((int)fy + 32768) << 16)));
    }
    cell[q] = code;
  }
  __syncthreads();
  const int nvalid = nvalid_s;
  const float* g = grid + (size_t)env * G * G;
  // The 49 x 128 x 9 gathers of one environment hit the same 64 KB of grid about 3.4 times per cell, as scattered
  // 32-byte sectors (measured: the L1-missing gathers ran at the L2 sector rate, 0.65 ms per step at N = 4096):
  // stream the grid once, coalesced, into shared memory -- as occupancy probabilities, so the logistic is
  // evaluated once per cell (the same expression, the same bits) -- and gather from there.
  // Rows are padded by 8 words: a warp covers ~4.5 rows of 7 consecutive candidates, and rows a multiple of 32 words
  // apart would put them all on the same 7 banks.
  const int Gs = G + 8;
  if (occ_in_smem) {
    const float4* g4 = reinterpret_cast<const float4*>(g);
    const int G4 = G >> 2;
    for (int q = tid; q < G * G4; q += kLatThreads) {
      const float4 v = __ldg(g4 + q);
      const int row = q / G4, c4 = q - row * G4;
      reinterpret_cast<float4*>(occ + row * Gs)[c4] = make_float4(1.f / (1.f + __expf(-v.x)), 1.f / (1.f + __expf(-v.y)), 1.f / (1.f + __expf(-v.z)), 1.f / (1.f + __expf(-v.w)));
    }
    __syncthreads();
  }
  float b1 = -1.f, b2 = -1.f;
  int bi = 0x7fffffff;
  const int C = nt * ny * nx;
  for (int c = tid; c < C; c += kLatThreads) {
    const int it = c / (ny * nx), rem = c - it * ny * nx, iy = rem / nx, ix = rem - iy * nx;
    const int dx = (ix - p.hx) * m - 32768, dy = (iy - p.hy) * m - 32768;
    const int* cl = cell + (size_t)it * R;
    float sum = 0.f;
    for (int i = 0; i < R; ++i) {
      const int code = cl[i];
      int jx = (code & 0xffff) + dx, jy = (int)((unsigned)code >> 16) + dy;
      if (code == 0) {   // edge ray: the general kernel's expression for this candidate
        const double cx = px + (double)((ix - p.hx) * p.sxy), cy = py + (double)((iy - p.hy) * p.sxy);
        const double* t = cs + ((size_t)it * R + i) * 2;
        jx = (int)floor((cx + t[0] - o) * ires);
        jy = (int)floor((cy + t[1] - o) * ires);
      }
      if ((unsigned)jx < (unsigned)G && (unsigned)jy < (unsigned)G)
        sum += occ_in_smem ? occ[jy * Gs + jx] : 1.f / (1.f + __expf(-__ldg(g + (size_t)jy * G + jx)));
    }
    const float sc = nvalid ? sum / (float)nvalid : 0.f;
    if (sc > b1) { b2 = b1; b1 = sc; bi = c; }      // candidates visited in increasing index: ties keep the lowest
    else if (sc > b2) b2 = sc;
  }
  // best / second best over the CTA: (b1, bi) = best with ties to the lowest index, b2 = best of all the others
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float o1 = __shfl_xor_sync(0xffffffffu, b1, off), o2 = __shfl_xor_sync(0xffffffffu, b2, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    const bool mine = b1 > o1 || (b1 == o1 && bi < oi);
    const float lose = mine ? o1 : b1;
    b1 = mine ? b1 : o1;
    bi = mine ? bi : oi;
    b2 = fmaxf(fmaxf(b2, o2), lose);
  }
  if (lane == 0) { w_b1[wid] = b1; w_b2[wid] = b2; w_bi[wid] = bi; }
  __syncthreads();
  if (tid == 0) {
    float g1 = w_b1[0], g2 = w_b2[0];
    int gi = w_bi[0];
    for (int k = 1; k < kLatThreads / 32; ++k) {
      const bool mine = g1 > w_b1[k] || (g1 == w_b1[k] && gi < w_bi[k]);
      const float lose = mine ? w_b1[k] : g1;
      g1 = mine ? g1 : w_b1[k];
      gi = mine ? gi : w_bi[k];
      g2 = fmaxf(fmaxf(g2, w_b2[k]), lose);
    }
    if (g2 < 0.f) g2 = 0.f;
    const int it = gi / (ny * nx), rem = gi - it * ny * nx, iy = rem / nx, ix = rem - iy * nx;
    pose_meas[env] = (float)(px + (double)((ix - p.hx) * p.sxy));
    pose_meas[(size_t)N + env] = (float)(py + (double)((iy - p.hy) * p.sxy));
    pose_meas[2 * (size_t)N + env] = (float)(pth + (double)((it - p.ht) * p.sth));
    score[env] = g1;
    second[env] = g2;
  }
}

// one thread per ray: Amanatides-Woo traversal in fp64 (integer decisions, same operations as the oracle)
__global__ void __launch_bounds__(kThreads) grid_update_kernel(slam_scan_params p, int N, float* grid, const float* __restrict__ pose,
                                                                const float* __restrict__ ranges,
                                                                const float* __restrict__ weight, float l_free, float l_occ) {
  const int env = blockIdx.x, G = p.G;
  const double x0 = (double)pose[env], y0 = (double)pose[(size_t)N + env], th = (double)pose[2 * (size_t)N + env];
  const float w = weight[env];
  float* g = grid + (size_t)env * G * G;
  const double res = (double)p.res, o = -0.5 * G * res;
  for (int i = threadIdx.x; i < p.R; i += kThreads) {
    const float rf = ranges[(size_t)i * N + env];
    if (!(rf >= p.r_min && rf <= p.r_max)) continue;
    const double a = th + ray_angle(i, p.R), r = (double)rf;
    const double x1 = x0 + r * cos(a), y1 = y0 + r * sin(a);
    int ix = (int)floor((x0 - o) / res), iy = (int)floor((y0 - o) / res);
    const int jx = (int)floor((x1 - o) / res), jy = (int)floor((y1 - o) / res);
    const double dx = x1 - x0, dy = y1 - y0;
    const int sx = dx > 0 ? 1 : -1, sy = dy > 0 ? 1 : -1;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const double tdx = dx != 0 ? res / fabs(dx) : inf, tdy = dy != 0 ? res / fabs(dy) : inf;
    const double bx = o + (ix + (dx > 0 ? 1 : 0)) * res, by = o + (iy + (dy > 0 ? 1 : 0)) * res;
    double tmx = dx != 0 ? (bx - x0) / dx : inf, tmy = dy != 0 ? (by - y0) / dy : inf;
    const int n = abs(jx - ix) + abs(jy - iy);
    for (int k = 0; k <= n; ++k) {
      const bool last = ix == jx && iy == jy;
      if (ix >= 0 && ix < G && iy >= 0 && iy < G) atomicAdd(g + (size_t)iy * G + ix, last ? l_occ * w : -l_free * w);
      if (last) break;
      if (tmx < tmy) { tmx += tdx; ix += sx; }
      else { tmy += tdy; iy += sy; }
    }
  }
}

__global__ void grid_clamp_kernel(float* grid, size_t n, float l_clamp) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) grid[i] = fminf(fmaxf(grid[i], -l_clamp), l_clamp);
}

bool params_ok(const slam_scan_params* p, int batch) {
  return p && batch >= 1 && p->G >= 8 && p->G <= 2048 && p->R >= 2 && p->R <= 1024 && p->res > 0.f && p->r_max > p->r_min &&
         p->hx >= 0 && p->hy >= 0 && p->ht >= 0 && p->hx <= 32 && p->hy <= 32 && p->ht <= 32 && p->sxy > 0.f && p->sth > 0.f;
}

}  // namespace

extern "C" {

int slam_scan_match(const slam_scan_params* p, int batch, const float* grid, const float* pose_pred, const float* ranges,
                    float* pose_meas, float* score, float* second, void* stream) {
  if (!params_ok(p, batch) || !grid || !pose_pred || !ranges || !pose_meas || !score || !second) return SLAM_EINVAL;
  size_t smem = (size_t)(2 * p->ht + 1) * p->R * 2 * sizeof(double) + (size_t)((p->R + 3) & ~3) * sizeof(float);
  if (smem > 100 * 1024) return SLAM_EINVAL;
  // lattice variant when the xy step is a whole number of cells (SLAM_SCAN_LATTICE=0 forces the general kernel)
  {
    const double q = (double)p->sxy / (double)p->res;
    const int m = (int)(q + 0.5);
    const char* el = getenv("SLAM_SCAN_LATTICE");
    if (m >= 1 && m <= 64 && (double)p->sxy == (double)m * (double)p->res && !(el && el[0] == '0')) {
      size_t smem_l = smem + (size_t)(2 * p->ht + 1) * p->R * sizeof(int);
      const size_t occ_b = (size_t)p->G * (p->G + 8) * sizeof(float);
      const char* es = getenv("SLAM_SCAN_SMEM");       // (the grid must be a whole number of float4, 16-byte aligned rows)
      const int occ_l = !(es && es[0] == '0') && (p->G & 3) == 0 && (((2 * p->ht + 1) * p->R) & 3) == 0 && smem_l + occ_b <= 110 * 1024 && ((uintptr_t)grid & 15) == 0;
      if (occ_l) smem_l += occ_b;
      if (cudaFuncSetAttribute(scan_match_lattice_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_l) != cudaSuccess) {
        cudaGetLastError();
        return SLAM_ECUDA;
      }
      const int C = (2 * p->ht + 1) * (2 * p->hy + 1) * (2 * p->hx + 1);
      const int threads = C >= kLatMax ? kLatMax : ((C + 31) / 32) * 32;
      scan_match_lattice_kernel<<<batch, threads, smem_l, (cudaStream_t)stream>>>(*p, batch, m, grid, pose_pred, ranges, pose_meas,
                                                                                      score, second, occ_l);
      return cudaGetLastError() == cudaSuccess ? SLAM_OK : SLAM_ECUDA;
    }
  }
  const size_t occ_bytes = (size_t)p->G * p->G * sizeof(float);
  // Measured on B200 (N = 4096, G = 128): staging the occupancy probabilities in shared memory is SLOWER
  // (2.31 ms vs 1.31 ms per step): it costs occupancy and random bank conflicts, while the L1-cached global
  // gathers of the 64 KB grid hit.  Kept behind SLAM_SCAN_SMEM=1 for larger rays-per-cell ratios.
  const char* e = getenv("SLAM_SCAN_SMEM");
  const int occ_in_smem = e && e[0] == '1' && smem + occ_bytes <= 110 * 1024;
  if (occ_in_smem) smem += occ_bytes;
  if (cudaFuncSetAttribute(scan_match_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
    cudaGetLastError();
    return SLAM_ECUDA;
  }
  scan_match_kernel<<<batch, kThreads, smem, (cudaStream_t)stream>>>(*p, batch, grid, pose_pred, ranges, pose_meas, score, second,
                                                                     occ_in_smem);
  return cudaGetLastError() == cudaSuccess ? SLAM_OK : SLAM_ECUDA;
}

int slam_grid_update(const slam_scan_params* p, int batch, float* grid, const float* pose, const float* ranges, const float* weight,
                     float l_free, float l_occ, float l_clamp, void* stream) {
  if (!params_ok(p, batch) || !grid || !pose || !ranges || !weight || !(l_clamp > 0.f)) return SLAM_EINVAL;
  grid_update_kernel<<<batch, kThreads, 0, (cudaStream_t)stream>>>(*p, batch, grid, pose, ranges, weight, l_free, l_occ);
  const size_t n = (size_t)batch * p->G * p->G;
  grid_clamp_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(grid, n, l_clamp);
  return cudaGetLastError() == cudaSuccess ? SLAM_OK : SLAM_ECUDA;
}

}  // extern "C"
