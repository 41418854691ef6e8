// wigner_seitz.cuh -- SURVEY 8(f) NEXT-3: Wigner-Seitz defect count.
//
// "The interstitials and vacancies were identified by using the Wigner-Seitz cell methods [34]":
// every atom is assigned to the reference lattice site nearest to it (minimum image on periodic axes), i.e.
// to the Wigner-Seitz cell it sits in; a site with no atom is a vacancy, a site holding m >= 2 atoms carries
// m - 1 interstitials.  Ties go to the lowest site index (C-25).
//
// Data-parallel over atoms, integer/HBM-bound: the reference sites are binned once into a grid of cells of
// about 4 sites each (k_ws_bin / k_ws_scan / k_ws_place); k_ws_assign gives one thread per atom, scans the
// 27 cells around the atom in fp64 and widens the block ring by ring until the best distance found is
// provably smaller than the distance to every unscanned cell, so the result is the exact nearest site for
// any atom position (sputtered atoms far from the lattice included).  Occupancies are integer atomics
// (order-independent), so the counts are reproducible.
#pragma once
#include "common.cuh"

struct WsGrid {  // host-filled, passed by value
  double lo[3], L[3], w[3], inv_w[3];  // grid origin, box edge, cell width per axis
  int nc[3], pbc[3];
  int ncells;
};

__device__ __forceinline__ int ws_cell_1d(const WsGrid& g, int a, double x) {
  if (g.pbc[a]) x -= g.L[a] * floor(x / g.L[a]);
  int c = (int)floor((x - g.lo[a]) * g.inv_w[a]);
  return c < 0 ? 0 : (c >= g.nc[a] ? g.nc[a] - 1 : c);
}

// min / max site coordinate per axis (order-preserving integer encoding), for the grid on open axes
__global__ void __launch_bounds__(256)
k_ws_bounds(int ns, const double* __restrict__ site, unsigned long long* __restrict__ mnmx) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  for (int a = 0; a < 3; ++a) {
    double x = s < ns ? site[(size_t)a * ns + s] : 0.0;
    bool ok = s < ns && isfinite(x);
    unsigned long long kmin = ok ? enc_double(x) : ~0ull, kmax = ok ? enc_double(x) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      unsigned long long a1 = __shfl_xor_sync(0xffffffffu, kmin, o);
      unsigned long long a2 = __shfl_xor_sync(0xffffffffu, kmax, o);
      kmin = a1 < kmin ? a1 : kmin;
      kmax = a2 > kmax ? a2 : kmax;
    }
    if ((threadIdx.x & 31) == 0) {
      atomicMin(&mnmx[a], kmin);
      atomicMax(&mnmx[3 + a], kmax);
    }
  }
}

__global__ void __launch_bounds__(256)
k_ws_bin(const WsGrid g, int ns, const double* __restrict__ site, int* __restrict__ cell_of,
         int* __restrict__ cell_count) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= ns) return;
  int cx = ws_cell_1d(g, 0, site[s]), cy = ws_cell_1d(g, 1, site[(size_t)ns + s]),
      cz = ws_cell_1d(g, 2, site[2 * (size_t)ns + s]);
  int c = (cz * g.nc[1] + cy) * g.nc[0] + cx;
  cell_of[s] = c;
  atomicAdd(&cell_count[c], 1);
}

// exclusive scan of cell_count[0..ncells) -> cell_start[0..ncells]; one block of 1024 threads
__global__ void __launch_bounds__(1024)
k_ws_scan(int ncells, const int* __restrict__ cell_count, int* __restrict__ cell_start) {
  __shared__ int part[1024];
  int chunk = (ncells + 1023) / 1024;
  int b = min(threadIdx.x * chunk, ncells), e = min(b + chunk, ncells);
  int s = 0;
  for (int c = b; c < e; ++c) s += cell_count[c];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    int v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  int run = threadIdx.x ? part[threadIdx.x - 1] : 0;
  for (int c = b; c < e; ++c) {
    cell_start[c] = run;
    run += cell_count[c];
  }
  if (threadIdx.x == 1023) cell_start[ncells] = part[1023];
}

// sites in cell order as 32-byte records {x, y, z, index}: the assignment reads one record with ONE 256-bit
// load (the first version kept x, y, z, index in four arrays and was bound by the L1 wavefronts of four
// scattered loads per candidate: 102 us for 128 000 atoms).  The order inside a cell is the ticket order of
// the atomics; the assignment does not depend on it (ties are broken by site index).
struct __align__(32) WsSite {
  double x, y, z;
  int idx, pad;
};
__global__ void __launch_bounds__(256)
k_ws_place(int ns, const double* __restrict__ site, const int* __restrict__ cell_of,
           const int* __restrict__ cell_start, int* __restrict__ cell_fill, WsSite* __restrict__ rec) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= ns) return;
  int c = cell_of[s];
  int k = cell_start[c] + atomicAdd(&cell_fill[c], 1);
  WsSite r;
  r.x = site[s];
  r.y = site[(size_t)ns + s];
  r.z = site[2 * (size_t)ns + s];
  r.idx = s;
  r.pad = 0;
  rec[k] = r;
}
__device__ __forceinline__ void ws_load(const WsSite* p, double& x, double& y, double& z, int& idx) {
  unsigned v0, v1, v2, v3, v4, v5, v6, v7 = 0;
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3), "=r"(v4), "=r"(v5), "=r"(v6), "+r"(v7)
               : "l"(p));
  idx = (int)(v6 | (v7 & 0u));  // (the padding word is part of the 256-bit load)
  x = __hiloint2double((int)v1, (int)v0);
  y = __hiloint2double((int)v3, (int)v2);
  z = __hiloint2double((int)v5, (int)v4);
}

// One thread per atom: exact nearest reference site.  Distances are evaluated in fp64 with the same
// operations in the same order as the plain definition (d = site - pos; d -= L rint(d / L) on periodic
// axes; r2 = (dx^2 + dy^2) + dz^2, no FMA contraction), so the chosen index is the definition's.
// The atom's own cell is scanned first; another cell of the block is scanned only if the box of that cell
// comes closer to the atom than the best site found so far (with a 1e-9 safety margin for the rounding of
// the cell geometry), which leaves ~10 candidates per atom of a crystal instead of the ~108 of all 27 cells
// (the kernel is instruction-bound: ncu, profiles/).
// latency-bound (three dependent loads, fp64 chains): 12 blocks per SM at 40 registers -- 0.71 ms (72 registers,
// 7 blocks) -> 0.54 ms per count at 8.192 M atoms; 16 blocks at 32 registers 0.57 ms
__global__ void __launch_bounds__(128, 12)
k_ws_assign(const WsGrid g, int n, const double* __restrict__ pos, const int* __restrict__ cell_start,
            const WsSite* __restrict__ rec, int* __restrict__ nearest, int* __restrict__ occ) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double p[3] = {pos[i], pos[(size_t)n + i], pos[2 * (size_t)n + i]};
  if (!(isfinite(p[0]) && isfinite(p[1]) && isfinite(p[2]))) {
    if (nearest) nearest[i] = -1;
    return;
  }
  int c[3];
  double fa[3];  // coordinate of the atom relative to the lower face of its cell (outside [0, w) only for
                 // atoms beyond the grid on open axes, which are binned into the boundary cell)
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    c[a] = ws_cell_1d(g, a, p[a]);
    double x = p[a];
    if (g.pbc[a]) x -= g.L[a] * floor(x / g.L[a]);
    fa[a] = (x - g.lo[a]) - c[a] * g.w[a];
  }
  const double hL[3] = {0.5 * g.L[0], 0.5 * g.L[1], 0.5 * g.L[2]};
  double best = INFINITY;
  int bs = 0x7fffffff;
  auto scan_cell = [&](int cell) {
    const int b = cell_start[cell], e = cell_start[cell + 1];
    for (int k = b; k < e; ++k) {
      double qx, qy, qz;
      int s;
      ws_load(rec + k, qx, qy, qz, s);
      double d0 = qx - p[0], d1 = qy - p[1], d2 = qz - p[2];
      // |d| <= L/2  =>  rint(d / L) == 0 (correctly rounded division is monotone, halves round to
      // even) and d - L * 0 == d: skipping the fp64 division there leaves every bit unchanged
      if (g.pbc[0] && fabs(d0) > hL[0]) d0 = __dsub_rn(d0, __dmul_rn(g.L[0], rint(d0 / g.L[0])));
      if (g.pbc[1] && fabs(d1) > hL[1]) d1 = __dsub_rn(d1, __dmul_rn(g.L[1], rint(d1 / g.L[1])));
      if (g.pbc[2] && fabs(d2) > hL[2]) d2 = __dsub_rn(d2, __dmul_rn(g.L[2], rint(d2 / g.L[2])));
      double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d0, d0), __dmul_rn(d1, d1)), __dmul_rn(d2, d2));
      if (r2 < best || (r2 == best && s < bs)) {
        best = r2;
        bs = s;
      }
    }
  };
  // distance along axis a from the atom to the cell at offset o from its own cell (0 if it overlaps)
  auto axis_gap = [&](int a, int o) -> double {
    double lo = o * g.w[a] - fa[a], hi = lo + g.w[a];
    return lo > 0.0 ? lo : (hi < 0.0 ? -hi : 0.0);
  };
  scan_cell((c[2] * g.nc[1] + c[1]) * g.nc[0] + c[0]);
  // R = 1 (27 cells) settles every atom of a crystal; a wider block is walked again whole (rare).
  // The 26 neighbour cells of R = 1 are almost all REJECTED by the gap test, so that test comes first and alone: the
  // nine squared axis gaps are formed once, a rejected cell costs two additions and a compare, the periodic wrap and
  // the cell index are computed for the accepted ones only (the general loop below spent ~40 instructions per
  // rejected cell: 0.92 ms per count at 8.192 M atoms, ncu).  Same gaps, same sums, same comparisons as below.
  int R0 = 1;
  if ((!g.pbc[0] || g.nc[0] >= 4) && (!g.pbc[1] || g.nc[1] >= 4) && (!g.pbc[2] || g.nc[2] >= 4)) {
    double g2[3][3];
    bool in[3][3];  // the cell at offset o - 1 exists (open axes end at the grid)
    bool all_covered = true;
    double bound = INFINITY;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
#pragma unroll
      for (int o = 0; o < 3; ++o) {
        const double gp = axis_gap(a, o - 1);
        g2[a][o] = gp * gp;
        in[a][o] = g.pbc[a] || (c[a] + o - 1 >= 0 && c[a] + o - 1 <= g.nc[a] - 1);
      }
      const bool covered = !g.pbc[a] && c[a] - 1 <= 0 && c[a] + 1 >= g.nc[a] - 1;
      if (!covered) bound = fmin(bound, g.w[a]);
      all_covered = all_covered && covered;
    }
    // which of the 26 cells can hold a site that beats or ties the best of the own cell (a later scan can only lower
    // the best: the set is a superset of what the general loop would scan, the result is the same)
    const double thr = best * (1.0 + 1e-9) + 1e-9;
    unsigned accept = 0u;
#pragma unroll
    for (int oz = 0; oz < 3; ++oz) {
#pragma unroll
      for (int oy = 0; oy < 3; ++oy) {
        const double gyz = g2[1][oy] + g2[2][oz];
#pragma unroll
        for (int ox = 0; ox < 3; ++ox) {
          if (ox == 1 && oy == 1 && oz == 1) continue;  // own cell: scanned above
          const double dmin2 = g2[0][ox] + gyz;
          if (!(dmin2 > thr) && in[0][ox] && in[1][oy] && in[2][oz]) accept |= 1u << ((oz * 3 + oy) * 3 + ox);
        }
      }
    }
    while (accept) {
      const int bit = __ffs((int)accept) - 1;
      accept &= accept - 1u;
      const int oz = bit / 9, oy = (bit / 3) % 3, ox = bit % 3;
      int cx = c[0] + ox - 1, cy = c[1] + oy - 1, cz = c[2] + oz - 1;
      if (g.pbc[0]) cx = cx < 0 ? cx + g.nc[0] : (cx >= g.nc[0] ? cx - g.nc[0] : cx);
      if (g.pbc[1]) cy = cy < 0 ? cy + g.nc[1] : (cy >= g.nc[1] ? cy - g.nc[1] : cy);
      if (g.pbc[2]) cz = cz < 0 ? cz + g.nc[2] : (cz >= g.nc[2] ? cz - g.nc[2] : cz);
      scan_cell((cz * g.nc[1] + cy) * g.nc[0] + cx);
    }
    R0 = (best < bound * bound || all_covered) ? 0 : 2;  // 0: settled
  }
  for (int R = R0; R > 0; ++R) {
    int lo[3], hi[3], covered[3];
    double bound = INFINITY;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = c[a] - R;
      hi[a] = c[a] + R;
      if (g.pbc[a]) {
        covered[a] = 2 * R + 1 >= g.nc[a];
        if (covered[a]) { lo[a] = 0; hi[a] = g.nc[a] - 1; }
      } else {
        if (lo[a] < 0) lo[a] = 0;
        if (hi[a] > g.nc[a] - 1) hi[a] = g.nc[a] - 1;
        covered[a] = lo[a] == 0 && hi[a] == g.nc[a] - 1;
      }
      // a site in a cell outside the block along this axis is at least R cell widths away along it
      if (!covered[a]) bound = fmin(bound, R * g.w[a]);
    }
    for (int vz = lo[2]; vz <= hi[2]; ++vz) {
      int cz = vz;
      if (g.pbc[2] && !covered[2]) cz = vz < 0 ? vz + g.nc[2] : (vz >= g.nc[2] ? vz - g.nc[2] : vz);
      const double gz = (g.pbc[2] && covered[2]) ? 0.0 : axis_gap(2, vz - c[2]);
      for (int vy = lo[1]; vy <= hi[1]; ++vy) {
        int cy = vy;
        if (g.pbc[1] && !covered[1]) cy = vy < 0 ? vy + g.nc[1] : (vy >= g.nc[1] ? vy - g.nc[1] : vy);
        const double gy = (g.pbc[1] && covered[1]) ? 0.0 : axis_gap(1, vy - c[1]);
        const double gyz = gy * gy + gz * gz;
        for (int vx = lo[0]; vx <= hi[0]; ++vx) {
          int cx = vx;
          if (g.pbc[0] && !covered[0]) cx = vx < 0 ? vx + g.nc[0] : (vx >= g.nc[0] ? vx - g.nc[0] : vx);
          const double gx = (g.pbc[0] && covered[0]) ? 0.0 : axis_gap(0, vx - c[0]);
          const double dmin2 = gx * gx + gyz;
          if (dmin2 > best * (1.0 + 1e-9) + 1e-9) continue;  // no site of this cell can beat or tie the best
          if (R == 1 && cx == c[0] && cy == c[1] && cz == c[2]) continue;  // own cell: scanned above
          scan_cell((cz * g.nc[1] + cy) * g.nc[0] + cx);
        }
      }
    }
    if (best < bound * bound || (covered[0] && covered[1] && covered[2])) break;
  }
  if (bs == 0x7fffffff) bs = -1;  // no reference sites at all
  if (nearest) nearest[i] = bs;
  if (bs >= 0) atomicAdd(&occ[bs], 1);
}

// out[0] = number of sites with no atom (vacancies), out[1] = sum over sites of max(occ - 1, 0)
// (interstitials); integer atomics, order-independent
__global__ void __launch_bounds__(256)
k_ws_count(int ns, const int* __restrict__ occ, unsigned long long* __restrict__ out) {
  unsigned long long v = 0, q = 0;
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < ns; s += gridDim.x * blockDim.x) {
    int o = occ[s];
    v += o == 0;
    q += o > 1 ? (unsigned long long)(o - 1) : 0ull;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v += __shfl_xor_sync(0xffffffffu, v, o);
    q += __shfl_xor_sync(0xffffffffu, q, o);
  }
  if ((threadIdx.x & 31) == 0) {
    if (v) atomicAdd(&out[0], v);
    if (q) atomicAdd(&out[1], q);
  }
}
