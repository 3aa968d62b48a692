"""fp64 ORACLE of the paper's correlative scan matcher and occupancy-grid update (NEXT-3) -- TEST
INFRASTRUCTURE ONLY.  Plain numpy / Python loops, one environment at a time.

Paper: "a discretized neighborhood in (dx, dy, dtheta) is evaluated against the log-odds occupancy
grid.  The best-scoring candidate provides an absolute pose measurement, whose information matrix is
scaled according to the normalized match score and the ambiguity margin between the best and
second-best candidates"; "the aligned scan is integrated into the occupancy grid
using a confidence-dependent update weight proportional to the scan-matching score";
2D log-odds grid; 128 rays over 180 degrees, 0.1-10 m.  Everything
else is silent; the readings R28-R34 of DESIGN.md are restated at each step below.

Pins (tests/test_scanmatch.py): exact recovery of a lattice offset on a synthetic world, score = 1 on
a saturated map, symmetry of the candidate lattice, DDA cell sets against brute-force ray sampling,
conservation / sign of the grid update.
"""
import math

import numpy as np


def ray_angles(R):
    """R29: R rays over 180 degrees, phi_i = -pi/2 + i * pi / (R - 1)."""
    return -0.5 * math.pi + np.arange(R) * (math.pi / (R - 1))


def cell_of(x, y, G, res):
    """R28: square G x G grid centred on the world origin; cell (ix, iy) covers
    [ox + ix res, ox + (ix+1) res) with ox = -G res / 2.  Returns (ix, iy) (may be out of range)."""
    o = -0.5 * G * res
    return int(math.floor((x - o) / res)), int(math.floor((y - o) / res))


def candidates(hx, hy, ht, sxy, sth):
    """R30: offsets in GLOBAL axes; index = (it (2hy+1) + iy) (2hx+1) + ix."""
    out = []
    for it in range(2 * ht + 1):
        for iy in range(2 * hy + 1):
            for ix in range(2 * hx + 1):
                out.append(((ix - hx) * sxy, (iy - hy) * sxy, (it - ht) * sth))
    return out


def score(grid, pose, ranges, res, r_min, r_max):
    """R31: mean occupancy probability 1/(1+exp(-l)) of the cells hit by the valid ray end points;
    end points outside the grid contribute 0; no valid ray -> 0."""
    G = grid.shape[0]
    phi = ray_angles(len(ranges))
    total, nvalid = 0.0, 0
    for i, r in enumerate(ranges):
        if not (r_min <= r <= r_max):
            continue
        nvalid += 1
        ex = pose[0] + r * math.cos(pose[2] + phi[i])
        ey = pose[1] + r * math.sin(pose[2] + phi[i])
        ix, iy = cell_of(ex, ey, G, res)
        if 0 <= ix < G and 0 <= iy < G:
            total += 1.0 / (1.0 + math.exp(-grid[iy, ix]))
    return total / nvalid if nvalid else 0.0


def scan_match(grid, pose_pred, ranges, res, hx, hy, ht, sxy, sth, r_min=0.1, r_max=10.0):
    """Returns (pose_meas[3], best score, second-best score, best index, all scores).  R32: ties go to
    the lowest candidate index; the second-best is the best of the other candidates."""
    cands = candidates(hx, hy, ht, sxy, sth)
    sc = np.array([score(grid, (pose_pred[0] + dx, pose_pred[1] + dy, pose_pred[2] + dt), ranges, res, r_min, r_max)
                   for dx, dy, dt in cands])
    best = int(np.argmax(sc))
    others = np.delete(sc, best)
    second = float(others.max()) if len(others) else 0.0
    dx, dy, dt = cands[best]
    return np.array([pose_pred[0] + dx, pose_pred[1] + dy, pose_pred[2] + dt]), float(sc[best]), second, best, sc


def traverse(x0, y0, x1, y1, G, res):
    """R34: cells crossed by the segment from (x0,y0) to (x1,y1), in order, by the integer DDA of
    Amanatides & Woo (each cell once); cells outside the grid are skipped.  The last cell is the one
    that contains the end point."""
    o = -0.5 * G * res
    ix, iy = int(math.floor((x0 - o) / res)), int(math.floor((y0 - o) / res))
    jx, jy = int(math.floor((x1 - o) / res)), int(math.floor((y1 - o) / res))
    dx, dy = x1 - x0, y1 - y0
    sx = 1 if dx > 0 else -1
    sy = 1 if dy > 0 else -1
    tdx = res / abs(dx) if dx != 0 else math.inf
    tdy = res / abs(dy) if dy != 0 else math.inf
    bx = o + (ix + (1 if dx > 0 else 0)) * res
    by = o + (iy + (1 if dy > 0 else 0)) * res
    tmx = (bx - x0) / dx if dx != 0 else math.inf
    tmy = (by - y0) / dy if dy != 0 else math.inf
    cells = []
    n = abs(jx - ix) + abs(jy - iy)
    for _ in range(n + 1):
        if 0 <= ix < G and 0 <= iy < G:
            cells.append((ix, iy))
        if ix == jx and iy == jy:
            break
        if tmx < tmy:
            tmx += tdx
            ix += sx
        else:
            tmy += tdy
            iy += sy
    return cells


def grid_update(grid, pose, ranges, weight, res, l_free, l_occ, l_clamp, r_min=0.1, r_max=10.0):
    """R34: every valid ray adds -l_free*w to the cells it crosses before its end cell and +l_occ*w to
    the end cell; contributions are summed first, the result is clamped to [-l_clamp, l_clamp]."""
    G = grid.shape[0]
    out = grid.astype(np.float64).copy()
    phi = ray_angles(len(ranges))
    for i, r in enumerate(ranges):
        if not (r_min <= r <= r_max):
            continue
        ex = pose[0] + r * math.cos(pose[2] + phi[i])
        ey = pose[1] + r * math.sin(pose[2] + phi[i])
        cells = traverse(pose[0], pose[1], ex, ey, G, res)
        jx, jy = cell_of(ex, ey, G, res)
        for (cx, cy) in cells:
            if cx == jx and cy == jy:
                out[cy, cx] += l_occ * weight
            else:
                out[cy, cx] -= l_free * weight
    return np.clip(out, -l_clamp, l_clamp)
