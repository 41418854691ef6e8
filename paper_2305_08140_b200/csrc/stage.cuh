// stage.cuh -- neighbour TILES staged in shared memory for the gather kernels (north_star: "neighbour tiles staged in
// shared memory (TMA where it pays)").  An EXPERIMENT with a measured verdict (profiles/r2_*):
// selected with NEPZBL_STAGE=1 (plain coalesced copies) or 2 (1-D bulk copies, cp.async.bulk + mbarrier); default off.
//
// Atoms are stored cell-sorted, x fastest, so the cells a run of atoms can have neighbours in are a handful of
// (z, y) rows, each ONE contiguous range of xyzt.  A tile is 64 consecutive atoms (one block of k_radial); at every
// list rebuild k_tiles works out the tile's ranges from the cell grid (TileDesc) and rewrites the tile's list entries
// as 16-bit offsets into the staged copy (nl_loc), so that per step the block copies ~25 ranges of ~1.2 KB into
// shared memory and the per-pair loads become LDS instead of scattered 16-byte global gathers.  A tile whose ranges
// do not fit (dense core, very small boxes) keeps nranges = -1 and uses the global path.
#pragma once
#include "common.cuh"

#define STAGE_TILE 64      // atoms per tile = atoms per k_radial block (x RADIAL_LANES threads)
#define STAGE_MAXR 96      // ranges per tile
#define STAGE_CAP 3072     // staged atoms per tile: 48 KB of int4

struct TileDesc {
  int nranges;                      // -1: not staged
  int total;                        // staged atoms
  int start[STAGE_MAXR];            // first sorted index of each range
  unsigned short len[STAGE_MAXR];
  unsigned short off[STAGE_MAXR];   // offset of the range in the staged copy
};

// cells [lo, hi] of one axis widened by S with periodic wrap / open clipping: up to two segments (inclusive)
__device__ inline int widen_axis(int lo, int hi, int nc, int pbc, int S, bool full, int seg[2][2]) {
  if (full || hi - lo + 1 + 2 * S >= nc) {
    seg[0][0] = 0; seg[0][1] = nc - 1;
    return 1;
  }
  int a = lo - S, b = hi + S;
  if (!pbc) {
    seg[0][0] = a < 0 ? 0 : a; seg[0][1] = b > nc - 1 ? nc - 1 : b;
    return 1;
  }
  if (a < 0) { seg[0][0] = 0; seg[0][1] = b; seg[1][0] = a + nc; seg[1][1] = nc - 1; return 2; }   // ascending memory order
  if (b >= nc) { seg[0][0] = 0; seg[0][1] = b - nc; seg[1][0] = a; seg[1][1] = nc - 1; return 2; }
  seg[0][0] = a; seg[0][1] = b;
  return 1;
}

// One block (STAGE_TILE threads) per tile, at every list rebuild.
__global__ void __launch_bounds__(STAGE_TILE)
k_tiles(const Scalars* sc, const BoxMap* __restrict__ bm, int n, int npad, const int* __restrict__ perm,
        const int* __restrict__ cell_of, const int* __restrict__ cell_start, const int* __restrict__ nn_r,
        const int* __restrict__ nl_r, TileDesc* __restrict__ desc, unsigned short* __restrict__ nl_loc) {
  if (!sc->do_rebuild) return;
  __shared__ TileDesc d;
  const int s0 = blockIdx.x * STAGE_TILE;
  const int s1 = min(n, s0 + STAGE_TILE) - 1;
  if (threadIdx.x == 0) {
    const int ncx = bm->nc[0], ncy = bm->nc[1], ncz = bm->nc[2], S = bm->S;
    const int cf = cell_of[perm[s0]], cl = cell_of[perm[s1]];
    const int xf = cf % ncx, yf = (cf / ncx) % ncy, zf = cf / (ncx * ncy);
    const int xl = cl % ncx, yl = (cl / ncx) % ncy, zl = cl / (ncx * ncy);
    const bool one_plane = zf == zl, one_row = one_plane && yf == yl;
    int zs[2][2], ys[2][2], xs[2][2];
    const int nz = widen_axis(zf, zl, ncz, bm->pbc[2], S, false, zs);
    const int ny = widen_axis(yf, yl, ncy, bm->pbc[1], S, !one_plane, ys);
    const int nx = widen_axis(xf, xl, ncx, bm->pbc[0], S, !one_row, xs);
    int nr = 0, total = 0;
    bool fits = true;
    for (int a = 0; a < nz && fits; ++a)
      for (int cz = zs[a][0]; cz <= zs[a][1] && fits; ++cz)
        for (int b = 0; b < ny && fits; ++b)
          for (int cy = ys[b][0]; cy <= ys[b][1] && fits; ++cy)
            for (int c = 0; c < nx; ++c) {
              const int row = (cz * ncy + cy) * ncx;
              const int st = cell_start[row + xs[c][0]], en = cell_start[row + xs[c][1] + 1];
              if (en <= st) continue;
              if (nr > 0 && d.start[nr - 1] + d.len[nr - 1] == st && d.len[nr - 1] + (en - st) < 60000) {
                d.len[nr - 1] = (unsigned short)(d.len[nr - 1] + (en - st));  // contiguous with the previous range
              } else {
                if (nr == STAGE_MAXR) { fits = false; break; }
                d.start[nr] = st;
                d.len[nr] = (unsigned short)(en - st);
                d.off[nr] = (unsigned short)total;
                ++nr;
              }
              total += en - st;
              if (total > STAGE_CAP) { fits = false; break; }
            }
    d.nranges = fits ? nr : -1;
    d.total = fits ? total : 0;
  }
  __syncthreads();
  {  // the descriptor goes to global memory word by word
    const int* src = reinterpret_cast<const int*>(&d);
    int* dst = reinterpret_cast<int*>(desc + blockIdx.x);
    for (int k = threadIdx.x; k < (int)(sizeof(TileDesc) / 4); k += STAGE_TILE) dst[k] = src[k];
  }
  if (d.nranges < 0) return;
  const int s = s0 + threadIdx.x;
  if (s >= n) return;
  const int cnt = nn_r[s], nr = d.nranges;
  for (int e = 0; e < cnt; ++e) {
    const int j = nl_r[nl_at(e, s, npad)];
    int loc = 0;
    for (int r = 0; r < nr; ++r) {
      const unsigned rel = (unsigned)(j - d.start[r]);
      if (rel < (unsigned)d.len[r]) { loc = d.off[r] + (int)rel; break; }
    }
    nl_loc[(size_t)e * npad + s] = (unsigned short)loc;
  }
}

// ---- per-step staging of a tile into shared memory (called by all threads of the block; returns after the copy
//      is complete and visible).  MODE 1: plain coalesced copies, one warp per range; MODE 2: 1-D bulk copies.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int MODE>
__device__ __forceinline__ void stage_tile(const TileDesc* __restrict__ gd, const int4* __restrict__ xyzt, int4* s_xyzt,
                                           TileDesc* sd, unsigned long long* mbar) {
  {
    const int* src = reinterpret_cast<const int*>(gd);
    int* dst = reinterpret_cast<int*>(sd);
    if (threadIdx.x < 2) dst[threadIdx.x] = src[threadIdx.x];  // header first: nranges, total
  }
  if (MODE == 2 && threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int nr = sd->nranges;
  if (nr < 0) return;
  {  // the ranges themselves (only as many as are used)
    const int* gs = gd->start;
    for (int k = threadIdx.x; k < nr; k += blockDim.x) {
      sd->start[k] = gs[k];
      sd->len[k] = gd->len[k];
      sd->off[k] = gd->off[k];
    }
  }
  __syncthreads();
  if (MODE == 1) {
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (int r = w; r < nr; r += nw) {
      const int4* src = xyzt + sd->start[r];
      int4* dst = s_xyzt + sd->off[r];
      const int len = sd->len[r];
      for (int t = l; t < len; t += 32) dst[t] = src[t];
    }
    __syncthreads();
  } else {
    if (threadIdx.x == 0)
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(sd->total * 16)
                   : "memory");
    __syncthreads();
    if (threadIdx.x < nr) {
      const int r = threadIdx.x;
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                       smem_u32(s_xyzt + sd->off[r])),
                   "l"(xyzt + sd->start[r]), "r"((int)sd->len[r] * 16), "r"(smem_u32(mbar))
                   : "memory");
    }
    unsigned done = 0;
    while (!done) {
      asm volatile(
          "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
          : "=r"(done)
          : "r"(smem_u32(mbar))
          : "memory");
    }
  }
}
