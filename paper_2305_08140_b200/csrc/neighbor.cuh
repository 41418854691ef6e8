// neighbor.cuh -- S1 (state prep) and S2 (cell-list neighbour build) kernels.
//
// S2 (BASELINE.json north_star "cell-list neighbour build"; cutoffs P:106):
//   bin atoms into cells of edge >= (rc_radial+skin)/S (S = 2 when every periodic axis then holds >= 5
//   cells, else 1), canonical in-cell order (ascending caller index), then per atom walk the (2S+1)^3
//   surrounding cells (z, y, x ascending) and list every j with
//   r_ij < rc_radial+skin (radial list) and the subset r_ij < rc_angular+skin (angular list).
// Half-size cells are used for two reasons: fewer candidates per atom (342 instead of 590 in bcc W),
// and -- because the atoms are STORED in cell order, x fastest -- consecutive list entries are then
// mostly adjacent in memory, so the 4 lanes that share an atom in the force kernels gather from the
// same 128-byte lines (the force kernels are bound by L1 wavefronts of scattered gathers, profiles/).
// Every rebuild kernel early-exits unless Scalars::do_rebuild is set (the stream path enqueues the
// chain every step; the graph path puts it in an IF node).
// Determinism: integer atomics only (counts / slot tickets); the ticket order is erased by the
// per-cell sort, so the sorted order and the lists are reproducible bit for bit.
#pragma once
#include "common.cuh"

// ---------------------------------------------------------------- open-axis bounds
__global__ void k_bounds(Scalars* sc, int n, const double* __restrict__ pos, int open0, int open1,
                         int open2) {
  if (!sc->do_rebuild) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int open[3] = {open0, open1, open2};
  for (int a = 0; a < 3; ++a) {
    if (!open[a]) continue;
    double x = i < n ? pos[(size_t)a * n + i] : 0.0;
    bool ok = i < n && isfinite(x);
    unsigned long long kmin = ok ? enc_double(x) : ~0ull, kmax = ok ? enc_double(x) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      unsigned long long a1 = __shfl_xor_sync(0xffffffffu, kmin, o);
      unsigned long long a2 = __shfl_xor_sync(0xffffffffu, kmax, o);
      kmin = a1 < kmin ? a1 : kmin;
      kmax = a2 > kmax ? a2 : kmax;
    }
    if ((threadIdx.x & 31) == 0) {
      atomicMin(&sc->bmin[a], kmin);
      atomicMax(&sc->bmax[a], kmax);
    }
  }
}

__global__ void k_rebuild_begin(Scalars* sc) {
  if (!sc->do_rebuild) return;
  for (int a = 0; a < 3; ++a) {
    sc->bmin[a] = ~0ull;
    sc->bmax[a] = 0ull;
  }
  // overflow_radial / overflow_angular are NOT reset here: they stay set until the host has reported them
  // (check_device_flags -> k_clear_errors), so an overflow in the middle of an md_run chunk is not lost when
  // a later rebuild of the same chunk happens to fit
  sc->top2_bits = 0ull;
}

// Fixed-point grid and cell grid for cells of edge >= rcs * f / S.  Returns the number of cells, or
// -1 if a periodic axis cannot hold the 2S+1 distinct stencil cells that S == 2 needs.
__device__ long long make_grid(Scalars* sc, BoxMap* bm, const BoxHost& bh, int S, int f) {
  const double two32 = 4294967296.0;
  const double cw = bh.rcs * f / S;
  long long total = 1;
  for (int a = 0; a < 3; ++a) {
    bm->pbc[a] = bh.pbc[a];
    bm->L[a] = bh.L[a];
    double span, lo;
    int nc, ncv;
    if (bh.tri) {  // fractional coordinates: span 1, cells counted along the distance between the faces of axis a
      lo = 0.0;
      span = 1.0;
      nc = (int)floor(bh.hgt[a] / cw);
      if (S == 2 && nc < 5) return -1;
      if (f == 1 && nc < 2) sc->box_too_small = 1;
      if (nc < 1) nc = 1;
      ncv = nc;
    } else if (bh.pbc[a]) {
      lo = 0.0;
      span = bh.L[a];
      nc = (int)floor(bh.L[a] / cw);
      if (S == 2 && nc < 5) return -1;
      if (f == 1 && nc < 2) sc->box_too_small = 1;
      if (nc < 1) nc = 1;
      ncv = nc;
    } else {
      // open axis (SURVEY C-14): grid spans the atoms' bounding range plus margins of rcs; the 2^32
      // span is twice that, so int32 differences never wrap for real pairs.
      double mn = dec_double(sc->bmin[a]), mx = dec_double(sc->bmax[a]);
      if (!(mx >= mn)) { mn = 0.0; mx = 0.0; }
      double E = mx - mn, M = bh.rcs * f;
      ncv = (int)ceil(2.0 * (E + 2.0 * M) / cw);
      if (ncv < 2) ncv = 2;
      span = ncv * cw;
      lo = mn - M;
      nc = (int)floor((M + E) / cw) + 1;
      if (nc > ncv) nc = ncv;
    }
    bm->lo[a] = lo;
    bm->inv_h[a] = two32 / span;
    bm->h[a] = span / two32;
    bm->hf[a] = (float)(span / two32);
    bm->nc[a] = nc;
    bm->ncv[a] = ncv;
    total *= nc;
  }
  bm->tri = bh.tri;
  for (int k = 0; k < 9; ++k) {
    bm->H[k] = bh.H[k];
    bm->Hi[k] = bh.Hi[k];
    bm->hm[k] = bh.tri ? (float)(bh.H[k] / two32) : 0.0f;
  }
  if (!bh.tri) {
    bm->hm[0] = bm->hf[0];
    bm->hm[4] = bm->hf[1];
    bm->hm[8] = bm->hf[2];
  }
  return total;
}

// Choose the grid for this build (one thread): half-size cells (S = 2) if they fit, else full-size
// cells (S = 1); coarsen (f = 2, 4, ...) only if the cell arrays are too small for the volume.
__global__ void k_boxmap(Scalars* sc, BoxMap* bm, BoxHost bh) {
  if (!sc->do_rebuild) return;
  for (int S = 2; S >= 1; --S) {
    for (int f = 1; f <= (1 << 20); f *= 2) {
      long long total = make_grid(sc, bm, bh, S, f);
      if (total < 0) break;  // S = 2 does not fit this box: try S = 1
      if (total <= bh.ncell_cap) {
        bm->ncells = (int)total;
        bm->S = S;
        return;
      }
    }
  }
  bm->ncells = 1;  // unreachable for finite boxes; keeps the chain well-defined
  bm->S = 1;
}

__global__ void k_zero_cells(const Scalars* sc, const BoxMap* bm, int* cell_count, int* cell_fill,
                             int ncell_cap) {
  if (!sc->do_rebuild) return;
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c <= ncell_cap) {
    cell_count[c] = 0;
    if (c < ncell_cap) cell_fill[c] = 0;
  }
}

// S1 for a rebuild: fixed-point compute copy (caller order) + cell histogram.
__global__ void k_bin(Scalars* sc, const BoxMap* __restrict__ bm, int n,
                      const double* __restrict__ pos, const int32_t* __restrict__ types, int n_types,
                      int4* __restrict__ xyzt_tmp, int* __restrict__ cell_of, int* cell_count) {
  if (!sc->do_rebuild) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double x = pos[i], y = pos[(size_t)n + i], z = pos[2 * (size_t)n + i];
  if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
    sc->nonfinite = 1;
    x = y = z = 0.0;
  }
  unsigned int uu[3];
  fix_position(bm, x, y, z, uu);
  const unsigned int ux = uu[0], uy = uu[1], uz = uu[2];
  int cx = cell_of_u(ux, bm->ncv[0], bm->nc[0]);
  int cy = cell_of_u(uy, bm->ncv[1], bm->nc[1]);
  int cz = cell_of_u(uz, bm->ncv[2], bm->nc[2]);
  int c = (cz * bm->nc[1] + cy) * bm->nc[0] + cx;
  xyzt_tmp[i] = make_int4((int)ux, (int)uy, (int)uz, checked_type(sc, types, i, n_types));
  cell_of[i] = c;
  atomicAdd(&cell_count[c], 1);
}

// exclusive scan of cell_count[0..ncells) -> cell_start[0..ncells] in three launches over tiles of SCAN_TILE cells
// (1024 threads x 4 consecutive cells: coalesced): k_scan_sums (tile totals) -> k_scan_tiles (ONE block scans the
// totals: ncells / 4096 values) -> k_scan_apply (every tile scans itself from its offset).  The first version was one
// block walking the whole array: 1.38 ms for the 3 M cells of 8.192 M atoms, one SM's worth of bandwidth.
constexpr int SCAN_TILE = 4096;

// exclusive scan of the block's tile v[4] per thread (1024 threads); returns the offset of the thread's first cell
// inside the tile, *total = the tile total (the same value in every thread)
__device__ __forceinline__ int scan_tile_1024(const int v[4], int* wsum, int* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int mine = v[0] + v[1] + v[2] + v[3];
  int x = mine;  // inclusive scan over the warp
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += t;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  if (w == 0) {
    int y = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, y, o);
      if (lane >= o) y += t;
    }
    wsum[lane] = y;
  }
  __syncthreads();
  *total = wsum[31];
  return (w ? wsum[w - 1] : 0) + x - mine;
}

__global__ void __launch_bounds__(1024) k_scan_sums(const Scalars* sc, const BoxMap* bm,
                                                    const int* __restrict__ cell_count, int* __restrict__ tile_sum) {
  if (!sc->do_rebuild) return;
  __shared__ int wsum[32];
  const int ncells = bm->ncells;
  const int c0 = blockIdx.x * SCAN_TILE + 4 * threadIdx.x;
  if (blockIdx.x * SCAN_TILE >= ncells) return;  // the grid is sized for the cell CAPACITY
  int v = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) v += c0 + k < ncells ? cell_count[c0 + k] : 0;
  v = __reduce_add_sync(0xffffffffu, v);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    v = __reduce_add_sync(0xffffffffu, wsum[threadIdx.x]);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = v;
  }
}

// one block: exclusive scan of the tile totals (in tiles of 4096 with a running carry; 733 values at 8.192 M atoms)
__global__ void __launch_bounds__(1024) k_scan_tiles(const Scalars* sc, const BoxMap* bm,
                                                     const int* __restrict__ tile_sum, int* __restrict__ tile_off) {
  if (!sc->do_rebuild) return;
  __shared__ int wsum[32];
  const int nt = (bm->ncells + SCAN_TILE - 1) / SCAN_TILE;
  int run = 0;  // totals before this round (the same value in every thread)
  for (int base = 0; base < nt; base += SCAN_TILE) {
    const int c0 = base + 4 * threadIdx.x;
    int v[4], total;
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = c0 + k < nt ? tile_sum[c0 + k] : 0;
    int off = run + scan_tile_1024(v, wsum, &total);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (c0 + k < nt) tile_off[c0 + k] = off;
      off += v[k];
    }
    run += total;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(1024) k_scan_apply(const Scalars* sc, const BoxMap* bm,
                                                     const int* __restrict__ cell_count,
                                                     const int* __restrict__ tile_off, int* __restrict__ cell_start) {
  if (!sc->do_rebuild) return;
  __shared__ int wsum[32];
  const int ncells = bm->ncells;
  if (blockIdx.x * SCAN_TILE >= ncells) return;
  const int c0 = blockIdx.x * SCAN_TILE + 4 * threadIdx.x;
  int v[4], total;
#pragma unroll
  for (int k = 0; k < 4; ++k) v[k] = c0 + k < ncells ? cell_count[c0 + k] : 0;
  const int base = tile_off[blockIdx.x];
  int off = base + scan_tile_1024(v, wsum, &total);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (c0 + k < ncells) cell_start[c0 + k] = off;
    off += v[k];
  }
  if ((blockIdx.x + 1) * SCAN_TILE >= ncells && threadIdx.x == 0) cell_start[ncells] = base + total;
}

__global__ void k_place(const Scalars* sc, int n, const int* __restrict__ cell_of,
                        const int* __restrict__ cell_start, int* cell_fill, int* __restrict__ order) {
  if (!sc->do_rebuild) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int c = cell_of[i];
  int t = atomicAdd(&cell_fill[c], 1);
  NZ_CHECK((unsigned)(cell_start[c] + t) < (unsigned)n, "k_place: slot outside [0, n)");
  order[cell_start[c] + t] = i;
}

// canonical in-cell order: ascending caller index (erases the ticket order of k_place)
__global__ void k_sortcell(const Scalars* sc, const BoxMap* bm, const int* __restrict__ cell_start,
                           int* __restrict__ order) {
  if (!sc->do_rebuild) return;
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= bm->ncells) return;
  int b = cell_start[c], e = cell_start[c + 1];
  for (int p = b + 1; p < e; ++p) {
    int v = order[p], q = p - 1;
    while (q >= b && order[q] > v) {
      order[q + 1] = order[q];
      --q;
    }
    order[q + 1] = v;
  }
}

__global__ void k_permute(const Scalars* sc, int n, const int* __restrict__ order,
                          const int4* __restrict__ xyzt_tmp, int* __restrict__ perm,
                          int* __restrict__ inv_perm, int4* __restrict__ xyzt,
                          int4* __restrict__ xyzt_build) {
  if (!sc->do_rebuild) return;
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int i = order[s];
  perm[s] = i;
  inv_perm[i] = s;
  int4 v = xyzt_tmp[i];
  xyzt[s] = v;
  xyzt_build[i] = v;  // CALLER order: k_kick_drift / k_prep read it coalesced, without waiting for inv_perm
}

// neighbour cells along one axis: up to 2S+1 distinct indices in out[0..2S], -1 = none
__device__ __forceinline__ void axis_stencil(int c, int nc, int pbc, int S, int out[5]) {
#pragma unroll
  for (int k = 0; k < 5; ++k) out[k] = -1;
  if (S == 2) {  // periodic axes hold >= 5 cells (k_boxmap), so the wrapped indices are distinct
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      int v = c + k - 2;
      if (pbc) {
        if (v < 0) v += nc;
        if (v >= nc) v -= nc;
      } else if (v < 0 || v >= nc) {
        v = -1;
      }
      out[k] = v;
    }
    return;
  }
  out[0] = c - 1;
  out[1] = c;
  out[2] = c + 1;
  if (pbc) {
    if (nc >= 3) {
      if (out[0] < 0) out[0] += nc;
      if (out[2] >= nc) out[2] -= nc;
    } else if (nc == 2) {
      out[0] = -1;             // c-1 and c+1 are the same cell
      out[2] = 1 - c;
    } else {
      out[0] = out[2] = -1;
    }
  } else {
    if (out[0] < 0) out[0] = -1;
    if (out[2] >= nc) out[2] = -1;
  }
}

// Runs of consecutive cells along x in walk order: the cells of a run are adjacent in the sorted atom array, so a
// run is ONE range of candidates (5 cells = ~13 atoms in bcc W instead of 5 ranges of ~2.7: a fifth of the
// cell_start look-ups and loop set-ups of the walk).  One run in the bulk, two where the stencil wraps around a
// periodic axis; the walk order (kz, ky, kx, then sorted index) is unchanged.
struct XRuns {
  int n, a[3], b[3];  // run r covers the x cells a[r] .. b[r]
};
__device__ __forceinline__ XRuns x_runs(const int sx[5], int W) {
  XRuns R;
  R.n = 0;
#pragma unroll
  for (int r = 0; r < 3; ++r) R.a[r] = R.b[r] = 0;
  int last = -2;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    if (k >= W || sx[k] < 0) continue;
    if (R.n > 0 && sx[k] == last + 1) {
#pragma unroll
      for (int r = 0; r < 3; ++r)
        if (r == R.n - 1) R.b[r] = sx[k];
    } else if (R.n < 3) {
#pragma unroll
      for (int r = 0; r < 3; ++r)
        if (r == R.n) R.a[r] = R.b[r] = sx[k];
      ++R.n;
    }
    last = sx[k];
  }
  return R;
}

// every candidate of atom s (sorted index) in walk order: f(j, r2).  The box matrix is read ONCE into registers (the
// first version went through fixed_disp_rt per candidate: four loads from the BoxMap and a branch in a 31-instruction
// test, ncu source page).
template <bool TRI, class F>
__device__ __forceinline__ void walk_candidates_t(const BoxMap* __restrict__ bm, int n, const int4* __restrict__ xyzt,
                                                  const int* __restrict__ cell_start, int s, const int4 me, int W,
                                                  const int sy[5], const int sz[5], const XRuns& R, F&& f) {
  float hm[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) hm[k] = (TRI || k % 4 == 0) ? bm->hm[k] : 0.0f;
  const int ncx = bm->nc[0], ncy = bm->nc[1];
  for (int kz = 0; kz < W; ++kz) {
    if (sz[kz] < 0) continue;
    for (int ky = 0; ky < W; ++ky) {
      if (sy[ky] < 0) continue;
      const int row = (sz[kz] * ncy + sy[ky]) * ncx;
      for (int r = 0; r < R.n; ++r) {
        const int ca = row + (r == 0 ? R.a[0] : r == 1 ? R.a[1] : R.a[2]);
        const int cb = row + (r == 0 ? R.b[0] : r == 1 ? R.b[1] : R.b[2]);
        NZ_CHECK((unsigned)ca < (unsigned)bm->ncells && (unsigned)cb < (unsigned)bm->ncells,
                 "k_nbr: stencil cell outside the grid");
        const int b = cell_start[ca], e = cell_start[cb + 1];
        NZ_CHECK(b >= 0 && b <= e && e <= n, "k_nbr: cell range outside [0, n]");
        for (int j = b; j < e; ++j) {  // j == s passes through: f rejects it (off the path of the ~73 % rejects)
          const int4 o = xyzt[j];
          float dx, dy, dz;  // int32 wrap-around = minimum image
          fixed_disp<TRI>(hm, o.x - me.x, o.y - me.y, o.z - me.z, dx, dy, dz);
          f(j, dx * dx + dy * dy + dz * dz);
        }
      }
    }
  }
}
template <class F>
__device__ __forceinline__ void walk_candidates(const BoxMap* __restrict__ bm, int n, const int4* __restrict__ xyzt,
                                                const int* __restrict__ cell_start, int s, const int4 me, int W,
                                                const int sy[5], const int sz[5], const XRuns& R, F&& f) {
  if (bm->tri) walk_candidates_t<true>(bm, n, xyzt, cell_start, s, me, W, sy, sz, R, f);
  else walk_candidates_t<false>(bm, n, xyzt, cell_start, s, me, W, sy, sz, R, f);
}

// per atom (sorted order): walk the (2S+1)^3 cells, emit ONE list (column-major) in three segments,
// each in walk order:
//   [0, nn_a)        pairs inside rc_angular + skin           -- this prefix IS the angular list
//   [nn_a, n_in)     the other pairs inside rc_radial at build time
//   [n_in, nn_r)     the pairs in the radial skin shell
// k_radial tests every entry against the true cutoffs each step; with this order the outcome is the
// same for almost all lanes of a warp, the in-cutoff entries k_force visits form a dense prefix, and
// the angular neighbours need no second list or second gather.  Two walks: the first counts the
// segments, the second places the entries (the cells are L1-hot by then).
__global__ void __launch_bounds__(128)
k_nbr(Scalars* sc, const BoxMap* __restrict__ bm, int n, int npad, const int4* __restrict__ xyzt,
      const int* __restrict__ cell_start, float rc2_radial, float rcs2_radial, float rcs2_angular, int cap_r, int cap_a,
      int* __restrict__ nn_r, int* __restrict__ nl_r, int* __restrict__ nn_a,
      unsigned long long* __restrict__ shellq, float rc_radial, float shell_w) {
  if (!sc->do_rebuild) return;
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const int4 me = xyzt[s];
  const int S = bm->S, W = 2 * S + 1;
  int sx[5], sy[5], sz[5];
  axis_stencil(cell_of_u((unsigned)me.x, bm->ncv[0], bm->nc[0]), bm->nc[0], bm->pbc[0], S, sx);
  axis_stencil(cell_of_u((unsigned)me.y, bm->ncv[1], bm->nc[1]), bm->nc[1], bm->pbc[1], S, sy);
  axis_stencil(cell_of_u((unsigned)me.z, bm->ncv[2], bm->nc[2]), bm->nc[2], bm->pbc[2], S, sz);
  const XRuns R = x_runs(sx, W);
  int na = 0, nb = 0, nc = 0;   // segment sizes
  unsigned long long shellq_val = ~0ull;  // "not ordered": set below when the shell could be sorted
  // ONE walk when the list fits the per-thread buffer (any cap_r <= NBR_BUF): the accepted candidates are parked,
  // tagged with their segment, in local memory and then laid out segment by segment; the first version walked the
  // cells twice and evaluated the ~340 candidate distances twice (k_nbr 1.54 ms at 1.024 M atoms).
  // The skin shell is laid out by SUB-SHELL (a counting sort over eight bins of width skin / 8, walk order inside a
  // bin), and shellq[s] keeps, byte m - 1, how many of its entries were put below rc + m * skin / 8.  An entry that lay
  // at r_b cannot be inside rc while the two largest displacements since the build add up to less than r_b - rc
  // (Scalars::disp_sum), so k_radial walks only the prefix of the shell that the current displacements can reach.
  // The bin of an entry is floor((r_b - rc) * 8 / skin - 1e-3): never ABOVE its true sub-shell (the 1e-3 covers the
  // approximate square root many times over), so the prefix of m bins holds every entry inside rc + m * skin / 8.
  // (The second version kept the distances beside the indices and insertion-sorted the shell: 1.5 KB of local memory
  // per thread, 160 MB in flight on the whole GPU -- more than the L2 -- and 25 GB of DRAM traffic per build at
  // 8.192 M atoms, ncu.)
  constexpr int NBR_BUF = 192;
  if (cap_r <= NBR_BUF) {
    int buf[NBR_BUF];
    int cnt = 0;
    unsigned long long binc = 0ull;  // entries per sub-shell, one byte each (a full list holds < 256 entries)
    const float inv_w = shell_w > 0.0f ? 1.0f / shell_w : 0.0f;
    walk_candidates(bm, n, xyzt, cell_start, s, me, W, sy, sz, R, [&](int j, float r2) {
      if (r2 < rcs2_radial && j != s) {
        const bool in_a = r2 < rcs2_angular, in_r = r2 < rc2_radial;
        const float fb = fmaf(r2, rsqrt_fast(r2), -rc_radial) * inv_w - 1e-3f;
        const int bin = min(max(__float2int_rd(fb), 0), 7);
        const int seg = in_a ? 0 : (in_r ? 1 : 2 + bin);
        na += in_a;
        nb += in_r && !in_a;
        if (!in_r) binc += 1ull << (8 * bin);
        if (cnt < NBR_BUF) buf[cnt] = j | (seg << 28);  // j < 2^28 (nep_zbl_set_workspace)
        ++cnt;
      }
    });
    nc = cnt - na - nb;
    if (!(cnt > cap_r || na > cap_a)) {
      // next slot of each segment: registers for the two inner ones, one byte per sub-shell of the skin shell
      int oa = 0, ob = na;
      const int oc = na + nb;
      unsigned long long pre = binc * 0x0101010101010100ull;  // exclusive prefix sums of the eight bytes
      shellq_val = binc * 0x0101010101010101ull;               // inclusive ones: byte m - 1 = entries below bin m
      for (int t = 0; t < cnt; ++t) {
        const int v = buf[t], seg = (unsigned)v >> 28;
        const int sh = 8 * max(seg - 2, 0);
        const int slot = seg == 0 ? oa : (seg == 1 ? ob : oc + (int)((pre >> sh) & 0xFFull));
        oa += seg == 0;
        ob += seg == 1;
        if (seg >= 2) pre += 1ull << sh;
        nl_r[nl_at(slot, s, npad)] = v & 0x0fffffff;
      }
    }
  } else {
  int oa = 0, ob = 0, oc = 0;   // next slot of each segment (second walk)
  for (int pass = 0; pass < 2; ++pass) {
    walk_candidates(bm, n, xyzt, cell_start, s, me, W, sy, sz, R, [&](int j, float r2) {
      if (r2 < rcs2_radial && j != s) {
        if (pass == 0) {
          if (r2 < rcs2_angular) ++na; else if (r2 < rc2_radial) ++nb; else ++nc;
        } else {
          int slot = r2 < rcs2_angular ? oa++ : (r2 < rc2_radial ? ob++ : oc++);
          nl_r[nl_at(slot, s, npad)] = j;
        }
      }
    });
    if (pass == 0) {
      if (na + nb + nc > cap_r || na > cap_a) break;  // overflow: reported below, nothing is written
      oa = 0;
      ob = na;
      oc = na + nb;
    }
  }
  }
  const int cr = na + nb + nc;
  if (shellq_val == ~0ull) {  // two-walk path or overflow: every sub-shell count = the whole shell (nothing is skipped)
    const unsigned long long c8 = (unsigned long long)min(nc, 255);
    shellq_val = c8 * 0x0101010101010101ull;
  }
  shellq[s] = shellq_val;
  nn_r[s] = min(cr, cap_r);
  nn_a[s] = (cr > cap_r || na > cap_a) ? 0 : na;
  if (cr > cap_r) atomicMax(&sc->overflow_radial, cr);
  if (na > cap_a) atomicMax(&sc->overflow_angular, na);
  if (cr > cap_r || na > cap_a) nn_r[s] = 0;
}

// reverse index of the (symmetric) angular list (the prefix [0, nn_a) of the list):
// rev[a][s] = position of s in the list of j = nl[a][s]
__global__ void k_rev(const Scalars* sc, int n, int npad, const int* __restrict__ nn_a,
                      const int* __restrict__ nl_a, unsigned char* __restrict__ rev) {
  if (!sc->do_rebuild) return;
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int na = nn_a[s];
  for (int a = 0; a < na; ++a) {
    int j = nl_a[nl_at(a, s, npad)];
    NZ_CHECK((unsigned)j < (unsigned)n, "k_rev: list entry outside [0, n)");
    // A list is in walk order = ascending sorted index unless j's stencil wraps around a periodic axis: bisect
    // (5 probes instead of ~13), and fall back to the plain search whenever the bisection does not land on s.
    // (Four bisections in flight per thread change nothing: the kernel moves 5.4 TB/s of sectors from the L2, the
    // column-major rows of 25 clusters of partners do not fit the L1.)
    const int nj = nn_a[j];
    int lo = 0, hi = nj;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (nl_a[nl_at(mid, j, npad)] < s) lo = mid + 1; else hi = mid;
    }
    int b = lo;
    if (!(b < nj && nl_a[nl_at(b, j, npad)] == s))
      for (b = 0; b < nj; ++b)
        if (nl_a[nl_at(b, j, npad)] == s) break;
    rev[(size_t)a * npad + s] = (unsigned char)(b < nj ? b : 255);
  }
}

// S1 for a plain evaluation: refresh the compute copy from caller positions (keeps the sorted
// order of the current list) and track the displacement since the build.
__global__ void __launch_bounds__(256)
k_prep(Scalars* sc, const BoxMap* __restrict__ bm, int n, const double* __restrict__ pos,
       const int32_t* __restrict__ types, int n_types, const int* __restrict__ inv_perm, int4* __restrict__ xyzt,
       const int4* __restrict__ xyzt_build) {
  __shared__ unsigned sh[64];
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.0f;
  if (i < n) {
    double x = pos[i], y = pos[(size_t)n + i], z = pos[2 * (size_t)n + i];
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
      sc->nonfinite = 1;
      x = y = z = 0.0;
    }
    unsigned int uu[3];
    fix_position(bm, x, y, z, uu);
    const unsigned int ux = uu[0], uy = uu[1], uz = uu[2];
    int s = inv_perm[i];
    int4 b = xyzt_build[i];
    xyzt[s] = make_int4((int)ux, (int)uy, (int)uz, checked_type(sc, types, i, n_types));
    float dx, dy, dz;
    fixed_disp_rt(bm, (int)ux - b.x, (int)uy - b.y, (int)uz - b.z, dx, dy, dz);
    d2 = dx * dx + dy * dy + dz * dz;
  }
  const Top2 m = block_top2(d2, sh);
  if (threadIdx.x == 0) top2_publish(&sc->top2_bits, m);
}

// decide whether the list must be rebuilt for this evaluation; reset per-evaluation counters.
__global__ void k_flag(Scalars* sc, float skin) {
  int r = sc->force_rebuild || top2_exceeds(sc->top2_bits, skin);
  sc->disp_sum = r ? 0.0f : top2_sum(sc->top2_bits);
  sc->top2_bits = 0ull;
  sc->do_rebuild = r;
  sc->force_rebuild = 0;
  sc->zbl_count = 0;
  sc->dense_count = 0;
  if (r) sc->n_rebuilds += 1;
}

// lists in the caller's indices, row-major [n][cap], -1 padded (neighbor_get)
__global__ void k_export_list(int n, int npad, int cap, const int* __restrict__ perm,
                              const int* __restrict__ nn, const int* __restrict__ nl,
                              int32_t* __restrict__ out_nn, int32_t* __restrict__ out_nl) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int i = perm[s], c = nn[s];
  out_nn[i] = c;
  for (int k = 0; k < cap; ++k)
    out_nl[(size_t)i * cap + k] = k < c ? perm[nl[nl_at(k, s, npad)]] : -1;
}
