// common.cuh -- device-side data layout of the NEP-ZBL hot path (sm_100a).
//
// Data layout in HBM:
//   master state   pos/vel fp64 SoA in the CALLER's atom order (caller-owned)
//   compute copy   xyzt[s] = {ux,uy,uz,type}: 32-bit FIXED-POINT coordinates (fraction of the box
//                  span per axis, 2^-32 units) in CELL-SORTED order s.  Differences of two such
//                  coordinates are exact integers and wrap modulo 2^32, i.e. the minimum image on
//                  periodic axes comes for free; resolution L/2^32 (1.2e-7 A at L = 506 A).
//   lists          column-major NL[slot][Npad] (coalesced over atoms), Npad = n rounded up to 128.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>

// Checked build (-DNEPZBL_CHECKED, libnepzbl_checked.so): every index that was read from memory and is about to be
// used as an address is tested against its bound; a violation prints where and traps (the launch fails loudly).
// compute-sanitizer is closed on the GPU pool this was developed on, so this is the memcheck stand-in: the GPU
// suite runs its small cases against the checked library (tests/test_gpu_checked.py).  No cost in the normal build.
#ifdef NEPZBL_CHECKED
#define NZ_CHECK(cond, what)                                                                                   \
  do {                                                                                                         \
    if (!(cond)) {                                                                                             \
      printf("nepzbl check failed: %s (%s:%d) block %d thread %d\n", what, __FILE__, __LINE__, (int)blockIdx.x, \
             (int)threadIdx.x);                                                                                \
      __trap();                                                                                                \
    }                                                                                                          \
  } while (0)
#else
#define NZ_CHECK(cond, what) do { } while (0)
#endif

#define NEPZBL_AMU_A2_FS2_TO_EV 103.6426965
#define NEPZBL_PI_F 3.14159265358979323846f

// 1 / sqrt(x) as the bare MUFU operation: rsqrtf() wraps it in a denormal fix-up (FMUL x 2^24, FSETP, FSEL, FMUL
// after) that squared pair distances of O(1 - 50 A^2) never need; x = 0 (coincident atoms) gives +inf either way
__device__ __forceinline__ float rsqrt_fast(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// 1 / x likewise (__fdividef adds a range check for huge denominators)
__device__ __forceinline__ float rcp_fast(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// The neighbour list nl[cap][npad] is stored with four consecutive entries of an atom side by side (an int4 per atom
// and group of four rows): the four lanes of an atom in k_radial / k_force read rows 4k .. 4k+3, so a warp's load of
// one entry per lane is ONE contiguous 128-byte line instead of four 32-byte sectors in four lines (the L1 data pipe is
// the second resource of those kernels, profiles/r2_ncu_full.md), and k_rev's bisection ends inside one sector.
__device__ __forceinline__ size_t nl_at(int row, int s, int npad) {
  return (((size_t)(row >> 2) * (size_t)npad + (size_t)s) << 2) + (size_t)(row & 3);
}

struct BoxMap {  // device-resident; recomputed by k_boxmap at every list rebuild
  double lo[3];     // origin of the fixed-point grid per axis
  double inv_h[3];  // 2^32 / span
  double h[3];      // span / 2^32   (Angstrom per unit)
  double L[3];      // box edge (periodic axes: span == L)
  float hf[3];
  int pbc[3];
  int nc[3];        // cells per axis actually used
  int ncv[3];       // cell index = (u * ncv) >> 32
  int ncells;
  int S;            // stencil half-width in cells: cells have edge >= (rc_radial+skin)/S
  // Triclinic boxes (C-28; all three axes periodic): the fixed-point coordinates are
  // the FRACTIONAL coordinates s = x H^-1 (H rows = lattice vectors), so integer differences still wrap to the
  // minimum image along every lattice vector; a difference (du_x, du_y, du_z) is the Cartesian vector
  // du_x hm[0..2] + du_y hm[3..5] + du_z hm[6..8], hm = H / 2^32.  Orthogonal boxes: tri = 0 and hm is diag(hf).
  int tri;
  double H[9], Hi[9];
  float hm[9];
};

// Cartesian displacement of an integer fixed-point difference
template <bool TRI>
__device__ __forceinline__ void fixed_disp(const float* __restrict__ hm, int dux, int duy, int duz, float& dx,
                                           float& dy, float& dz) {
  const float fx = (float)dux, fy = (float)duy, fz = (float)duz;
  if (TRI) {
    dx = fmaf(fz, hm[6], fmaf(fy, hm[3], fx * hm[0]));
    dy = fmaf(fz, hm[7], fmaf(fy, hm[4], fx * hm[1]));
    dz = fmaf(fz, hm[8], fmaf(fy, hm[5], fx * hm[2]));
  } else {
    dx = fx * hm[0];
    dy = fy * hm[4];
    dz = fz * hm[8];
  }
}
__device__ __forceinline__ void fixed_disp_rt(const BoxMap* __restrict__ bm, int dux, int duy, int duz, float& dx,
                                              float& dy, float& dz) {
  if (bm->tri) fixed_disp<true>(bm->hm, dux, duy, duz, dx, dy, dz);
  else fixed_disp<false>(bm->hm, dux, duy, duz, dx, dy, dz);
}

struct Scalars {  // device-resident control block (one per handle)
  int do_rebuild;
  int force_rebuild;
  unsigned long long top2_bits;         // float bits of the TWO largest |x_i - x_i(build)|^2 (hi word: largest)
  unsigned long long vmax2_bits[2];     // double bits: max_i |v_i|^2, double-buffered by step parity
  double dt;
  double dt_max, max_disp;              // md_step arguments (set by k_md_params)
  int parity;                           // which vmax2 slot holds max |v|^2 of the current state
  int trace_pos;                        // next slot of the dt trace ring
  unsigned long long bmin[3], bmax[3];  // order-preserving encodings of min/max coordinate (open axes)
  int overflow_radial, overflow_angular;  // largest neighbour counts seen since the host last cleared them
  int nonfinite;
  int box_too_small;
  int zbl_count;
  int dense_count;                      // atoms listed by k_angular_nn for the fp64 re-evaluation (site_fp64.cuh)
  int bad_type;                         // an atom type outside [0, n_types) was seen (clamped; reported as INVALID_ARG)
  int n_rebuilds;
  long long n_steps;
  float disp_sum;                       // d_(1) + d_(2) of the current positions against the build (0 right after a build)
  unsigned int blocks_done;             // ticket counter of k_kick_drift's last-block book-keeping
};

struct BoxHost {  // passed by value to k_boxmap
  double L[3];
  int pbc[3];
  double rcs;      // rc_radial + skin: minimum cell edge
  int ncell_cap;
  int tri;         // triclinic: H, Hi, hgt are set
  double H[9], Hi[9], hgt[3];  // lattice rows, inverse, distances between opposite faces
};

// order-preserving map double -> uint64 (for atomicMin/Max on signed doubles)
__host__ __device__ inline unsigned long long enc_double(double x) {
#ifdef __CUDA_ARCH__
  unsigned long long b = (unsigned long long)__double_as_longlong(x);
#else
  unsigned long long b;
  memcpy(&b, &x, 8);
#endif
  return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__device__ inline double dec_double(unsigned long long k) {
  unsigned long long b = (k & 0x8000000000000000ull) ? (k & 0x7fffffffffffffffull) : ~k;
  return __longlong_as_double((long long)b);
}

// atom type of atom i, validated: a type outside [0, n_types) would index the per-type tables (masses, atomic
// numbers, coefficient tables, records) out of bounds, so it is flagged (NEPZBL_E_INVALID_ARG) and replaced by 0
__device__ __forceinline__ int checked_type(Scalars* sc, const int32_t* __restrict__ types, int i, int n_types) {
  if (!types) return 0;
  const int t = types[i];
  if ((unsigned)t < (unsigned)n_types) return t;
  sc->bad_type = 1;
  return 0;
}

// fixed-point coordinate of x on one axis (wraps modulo 2^32 on periodic axes)
__device__ __forceinline__ unsigned int fix_coord(double x, double lo, double inv_h) {
  return (unsigned int)(unsigned long long)__double2ll_rd((x - lo) * inv_h);
}

// fixed-point coordinates of a Cartesian position: per axis for orthogonal boxes, fractional for triclinic ones
__device__ __forceinline__ void fix_position(const BoxMap* __restrict__ bm, double x, double y, double z,
                                             unsigned int u[3]) {
  if (bm->tri) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
      u[a] = fix_coord(x * bm->Hi[a] + y * bm->Hi[3 + a] + z * bm->Hi[6 + a], 0.0, 4294967296.0);
  } else {
    u[0] = fix_coord(x, bm->lo[0], bm->inv_h[0]);
    u[1] = fix_coord(y, bm->lo[1], bm->inv_h[1]);
    u[2] = fix_coord(z, bm->lo[2], bm->inv_h[2]);
  }
}

__device__ __forceinline__ int cell_of_u(unsigned int u, int ncv, int nc) {
  int c = (int)(((unsigned long long)u * (unsigned long long)ncv) >> 32);
  return c < nc ? c : nc - 1;
}

// Rebuild criterion (C-15): a pair inside the cutoff now was inside cutoff + skin at the build as long as
// d_i + d_j <= skin, and d_i + d_j <= d_(1) + d_(2), the two largest displacements since the build.  (The usual
// test d_(1) > skin / 2 is the special case d_(2) = d_(1); with ONE fast atom -- a primary knock-on -- the list
// lives twice as long.)  top-2 of squared displacements, kept as float bits (order-preserving for values >= 0).
struct Top2 {
  unsigned a, b;  // a >= b
};
__device__ __forceinline__ Top2 top2_merge(Top2 x, Top2 y) {
  Top2 r;
  r.a = max(x.a, y.a);
  r.b = max(min(x.a, y.a), max(x.b, y.b));
  return r;
}
// top-2 over a block of <= 1024 threads (one value per thread); result valid in thread 0
__device__ __forceinline__ Top2 block_top2(float v, unsigned* sh /* [64] */) {
  Top2 t{__float_as_uint(v), 0u};
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    Top2 u{__shfl_xor_sync(0xffffffffu, t.a, o), __shfl_xor_sync(0xffffffffu, t.b, o)};
    t = top2_merge(t, u);
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { sh[2 * w] = t.a; sh[2 * w + 1] = t.b; }
  __syncthreads();
  if (w == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    t.a = l < nw ? sh[2 * l] : 0u;
    t.b = l < nw ? sh[2 * l + 1] : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      Top2 u{__shfl_xor_sync(0xffffffffu, t.a, o), __shfl_xor_sync(0xffffffffu, t.b, o)};
      t = top2_merge(t, u);
    }
  }
  return t;
}
// Merge a block's top-2 into the global pair with two integer atomicMax (no CAS loop: ~500 blocks hit one address).
// W1 (high word) = largest: the exchange old = atomicMax(W1, a) has a loser min(old, a); W2 (low word) takes the
// maximum of all losers and of all blocks' second values.  Every loser is the smaller of two distinct atoms'
// values, so W2 never exceeds the true second largest, and the true second largest s is always recorded: when its
// block meets W1, either it loses at once (old >= s) or it wins and loses later to the one larger value.
__device__ __forceinline__ void top2_publish(unsigned long long* addr, Top2 t) {
  if (t.a == 0u) return;
  unsigned* w = reinterpret_cast<unsigned*>(addr);  // little endian: w[1] = largest, w[0] = second largest
  const unsigned old = atomicMax(&w[1], t.a);
  const unsigned second = max(min(old, t.a), t.b);
  if (second) atomicMax(&w[0], second);
}
// rebuild if the two largest displacements since the build add up to more than the skin (1e-5 safety margin for
// the rounding of the fixed-point differences and of sqrtf)
// upper bound of d_(1) + d_(2) (rounded up a little: it decides which skin-shell entries may be skipped)
__device__ __forceinline__ float top2_sum(unsigned long long bits) {
  return (sqrtf(__uint_as_float((unsigned)(bits >> 32))) + sqrtf(__uint_as_float((unsigned)bits))) * (1.0f + 1e-5f) + 1e-6f;
}
__device__ __forceinline__ int top2_exceeds(unsigned long long bits, float skin) {
  return sqrtf(__uint_as_float((unsigned)(bits >> 32))) + sqrtf(__uint_as_float((unsigned)bits)) > skin * (1.0f - 1e-5f);
}

__device__ __forceinline__ float block_max_128(float v, float* sh) {
  // max over a block of <= 1024 threads; result valid in thread 0
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) sh[w] = v;
  __syncthreads();
  if (w == 0) {
    int nw = (blockDim.x + 31) >> 5;
    v = l < nw ? sh[l] : 0.0f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  }
  return v;
}
