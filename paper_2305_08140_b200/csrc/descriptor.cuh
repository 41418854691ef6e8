// descriptor.cuh -- S3 (radial descriptor), S4 (angular descriptor), S6 (network) and the angular
// half of S7 (per-pair partial forces), one thread per atom in cell-sorted order.
//
// Formulas (the paper defers them to its ref. [25]; SURVEY 8(c) B-E is the reading):
//   f_c(r) = 1/2 [1 + cos(pi r / rc)],  x = 2 (r/rc - 1)^2 - 1,  f_k = 1/2 [T_k(x) + 1] f_c
//   g_n(r) = sum_k c_nk f_k(r)
//   q_n = sum_j g^R_n(r_ij);  q_nl = (2l+1)/(4 pi) sum_jk g^A_n g^A_n P_l(cos);  q^222_n (4-body)
//   U = sum_mu w1_mu tanh(sum_nu w0_mu,nu s_nu q_nu - b0_mu) - b1
// Factorisations used here (same numbers up to rounding):
//   * g_n = f_c * sum_k ct_nk T_k with ct folded on the host (ct_n0 = c_n0 + 1/2 sum_{k>=1} c_nk,
//     ct_nk = c_nk / 2), so q_n = sum_k ct_nk * (sum_j f_c T_k): the radial pass accumulates K
//     basis sums per atom instead of n_max*K products per neighbour (one atom type).
//   * 3-body by the addition theorem: q_nl = (2l+1)/(4 pi) sum_m C_lm A_nlm^2 with
//     A_nlm = sum_j g_n(r_ij) b_lm(rhat_ij), b_lm = real harmonic polynomials (unnormalised,
//     P_l^(m)(z) * Re/Im (x+iy)^m up to the scale folded into C_lm).
//   * 4-body: q^222_n = 3 C4 det S_n, S_n the traceless tensor rebuilt from the five l=2 sums.
//   * back-pass: dU_i/dr_ij = rhat S' + (v - rhat (rhat.v))/r with S' = sum_lm G'_lm b_lm,
//     v = sum_lm G_lm grad b_lm, G_lm = sum_n g_n E_nlm, G'_lm = sum_n g'_n E_nlm, E = dU/dA.
#pragma once
#include "common.cuh"
#include "stage.cuh"
#include "tc05.cuh"

template <int NR_, int KR_, int NA_, int KA_, bool B4_, int NT_ = 1, bool B5_ = false>
struct ModelShape {
  static constexpr int NT = NT_;  // atom types (2 = the type-pair tables c^{ti tj}_nk are exercised)
  static constexpr int NR = NR_;  // n_max_radial + 1
  static constexpr int KR = KR_;  // basis_radial + 1
  static constexpr int NA = NA_;
  static constexpr int KA = KA_;
  static constexpr bool B4 = B4_;
  static constexpr bool B5 = B5_;  // (1,1,1,1) 5-body term q_n = q_{n,l=1}^2 / 3 (C-27), behind the 4-body block
  static constexpr int LMAX = 4;
  static constexpr int NLM = 24;
  static constexpr int D = NR + NA * LMAX + (B4 ? NA : 0) + (B5 ? NA : 0);
  static constexpr int V5 = NR + NA * LMAX + (B4 ? NA : 0);  // first 5-body component
  static constexpr int DPAD = (D + 3) / 4 * 4;
  // record gathered per radial pair by k_force: {position, Fp[0..NR-1]} in ONE 32-byte sector when the
  // radial descriptor has at most 5 components, else {position, d[0..KR-1]} in 64 bytes (AtomRec)
  // (two atom types too: the neighbour's type then comes from k_radial's type mask, the type-pair table from shared memory)
  static constexpr bool FPREC = NR_ <= 5;
};

// Small tables passed by value (constant bank): compile-time indexed, so they cost no loads.
template <class MS>
struct ModelTables {
  // leading index: ordered type pair ti * NT + tj (central atom ti, neighbour tj)
  float ctR[MS::NT * MS::NT][MS::NR][MS::KR];   // folded radial coefficients
  float ctA[MS::NT * MS::NT][MS::NA][MS::KA];   // folded angular coefficients
  float kctA[MS::NT * MS::NT][MS::NA][MS::KA];  // k * ctA (derivative through T_k' = k U_{k-1})
  float inv_rcR, inv_rcA, rcR2, rcA2;
  float zbl_flag_r2;           // (r_outer + margin)^2, 0 if ZBL disabled
  float inv_shell_w;           // 8 / skin (0 without skin): sub-shells of the list's skin shell, see k_nbr
  float b1;
  int n_neurons;
  float dense_thr;             // 3-body network inputs |s q| above this send the atom to the fp64 pass (site_fp64.cuh)
  float dense_thr4;            // the same for the 4-body (and 5-body) inputs, whose fp32 error grows faster
};

// hand-over to the fp64 re-evaluation (site_fp64.cuh): atoms are appended to dense_list (integer ticket: the order
// of the list is free, every listed atom is evaluated on its own).  k_site_fp64 follows k_angular_nn as a plain
// kernel node that walks the list (measured on config2, where the list is empty: an IF node opened by k_angular_nn's
// last block cost 9.2 us per step, the plain node 5.5 us)
struct DenseArgs {
  Scalars* sc;
  int* dense_list;              // NULL: no listing
};

// Record of one atom for the radial back-pass of k_force (sorted order), 64-byte stride so that it
// never straddles a 128-byte line: {ux,uy,uz,d0..d4 | d5..d11 pad}.  d[k] = sum_n Fp[n] ct_nk are the
// atom's radial back-pass coefficients.  Fetched per pair with one 256-bit and one 128-bit load (two
// sectors of one line) -- k_force is bound by L1 tag lookups of scattered gathers when it gathers
// more, and by FP32 issue when it re-derives d from Fp per pair (both measured, profiles/).
struct __align__(64) AtomRec {
  int ux, uy, uz;  // fixed-point coordinates (same as xyzt)
  float d[12];     // d[0..KR-1]; rest zero
  float pad;
};
__device__ __forceinline__ void ld_rec(const AtomRec* p, int& ux, int& uy, int& uz, float d[12], int kr) {
  unsigned v0, v1, v2, v3, v4, v5, v6, v7;
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3), "=r"(v4), "=r"(v5), "=r"(v6), "=r"(v7)
               : "l"(p));
  ux = (int)v0; uy = (int)v1; uz = (int)v2;
  d[0] = __uint_as_float(v3); d[1] = __uint_as_float(v4); d[2] = __uint_as_float(v5);
  d[3] = __uint_as_float(v6); d[4] = __uint_as_float(v7);
  float4 t = __ldg(reinterpret_cast<const float4*>(p) + 2);
  d[5] = t.x; d[6] = t.y; d[7] = t.z; d[8] = t.w;
  if (kr > 9) {
    float4 u = __ldg(reinterpret_cast<const float4*>(p) + 3);
    d[9] = u.x; d[10] = u.y; d[11] = u.z;
  } else {
    d[9] = d[10] = d[11] = 0.0f;
  }
}
// atom type stored in the record's last word (models with more than one type)
__device__ __forceinline__ int ld_rec_type(const AtomRec* p) {
  return __float_as_int(__ldg(reinterpret_cast<const float*>(p) + 15));
}

// 32-byte record {ux,uy,uz,Fp0..Fp4} (ModelShape::FPREC): one sector, one 256-bit load per pair; the pair's
// coefficients d_i[k] + d_j[k] = sum_n (Fp_i[n] + Fp_j[n]) ct_nk are contracted in k_force (NR*KR FMAs with
// constant-bank operands) -- with the 64-byte record k_force was bound by the L1 data pipe (two scattered
// sector requests per pair, profiles/r1c_ncu_full.md).
__device__ __forceinline__ void ld_rec32(const void* base, int idx, int& ux, int& uy, int& uz, float f[5]) {
  const char* p = reinterpret_cast<const char*>(base) + (size_t)idx * 32;
  unsigned v0, v1, v2, v3, v4, v5, v6, v7;
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3), "=r"(v4), "=r"(v5), "=r"(v6), "=r"(v7)
               : "l"(p));
  ux = (int)v0; uy = (int)v1; uz = (int)v2;
  f[0] = __uint_as_float(v3); f[1] = __uint_as_float(v4); f[2] = __uint_as_float(v5);
  f[3] = __uint_as_float(v6); f[4] = __uint_as_float(v7);
}

// (2l+1)/(4 pi) * addition-theorem weight of each b_lm (see DESIGN.md for the list of b_lm)
__device__ __constant__ const float kClm[24] = {
    0.238732414637843f, 0.238732414637843f, 0.238732414637843f,                       // l=1: 3/(4pi)*{1,1,1}
    0.099471839432435f, 1.193662073189215f, 1.193662073189215f, 0.298415518297304f,
    0.298415518297304f,                                                                // l=2: 5/(4pi)*{1/4,3,3,3/4,3/4}
    0.139260575205408f, 0.208890862808112f, 0.208890862808112f, 2.088908628081126f,
    2.088908628081126f, 0.348151438013521f, 0.348151438013521f,                        // l=3: 7/(4pi)*{1/4,3/8,3/8,15/4,15/4,5/8,5/8}
    0.011190581936149f, 0.447623277445971f, 0.447623277445971f, 0.223811638722985f,
    0.223811638722985f, 3.133362942121796f, 3.133362942121796f, 0.391670367765225f,
    0.391670367765225f};                                                               // l=4: 9/(4pi)*{1/64,5/8,5/8,5/16,5/16,35/8,35/8,35/64,35/64}
#define NEPZBL_C4 (-0.269981309759908f) /* -45/(8 sqrt(14) pi^1.5) */

__device__ __forceinline__ int lm_to_l(int lm) { return lm < 3 ? 1 : (lm < 8 ? 2 : (lm < 15 ? 3 : 4)); }

// real harmonic polynomials of the unit vector (x,y,z), l = 1..4
__device__ __forceinline__ void eval_blm(float x, float y, float z, float b[24]) {
  float z2 = z * z, x2 = x * x, y2 = y * y;
  float c2 = x2 - y2, s2 = 2.0f * x * y;
  float c3 = x * (x2 - 3.0f * y2), s3 = y * (3.0f * x2 - y2);
  float c4 = c2 * c2 - s2 * s2, s4 = 2.0f * c2 * s2;
  float p31 = 5.0f * z2 - 1.0f, p41 = (7.0f * z2 - 3.0f) * z, p42 = 7.0f * z2 - 1.0f;
  b[0] = z; b[1] = x; b[2] = y;
  b[3] = 3.0f * z2 - 1.0f; b[4] = x * z; b[5] = y * z; b[6] = c2; b[7] = s2;
  b[8] = (5.0f * z2 - 3.0f) * z; b[9] = p31 * x; b[10] = p31 * y; b[11] = z * c2; b[12] = z * s2;
  b[13] = c3; b[14] = s3;
  b[15] = (35.0f * z2 - 30.0f) * z2 + 3.0f; b[16] = p41 * x; b[17] = p41 * y; b[18] = p42 * c2;
  b[19] = p42 * s2; b[20] = z * c3; b[21] = z * s3; b[22] = c4; b[23] = s4;
}

// S' = sum_lm Gp_lm b_lm and v = sum_lm G_lm grad_u b_lm (gradient of the polynomials in free x,y,z)
template <class F1, class F2>
__device__ __forceinline__ void contract_blm_grad(float x, float y, float z, F1 G, F2 Gp, float& Sp,
                                                  float& vx, float& vy, float& vz) {
  float z2 = z * z, x2 = x * x, y2 = y * y;
  float c2 = x2 - y2, s2 = 2.0f * x * y;
  float c3 = x * (x2 - 3.0f * y2), s3 = y * (3.0f * x2 - y2);
  float c4 = c2 * c2 - s2 * s2, s4 = 2.0f * c2 * s2;
  float p31 = 5.0f * z2 - 1.0f, p41 = (7.0f * z2 - 3.0f) * z, p42 = 7.0f * z2 - 1.0f;
  float xz = x * z, yz = y * z;
  float q41 = 21.0f * z2 - 3.0f;
  Sp = 0.0f; vx = 0.0f; vy = 0.0f; vz = 0.0f;
  float g;
  // l = 1
  Sp = fmaf(Gp(0), z, Sp); vz += G(0);
  Sp = fmaf(Gp(1), x, Sp); vx += G(1);
  Sp = fmaf(Gp(2), y, Sp); vy += G(2);
  // l = 2
  g = G(3); Sp = fmaf(Gp(3), 3.0f * z2 - 1.0f, Sp); vz = fmaf(g, 6.0f * z, vz);
  g = G(4); Sp = fmaf(Gp(4), xz, Sp); vx = fmaf(g, z, vx); vz = fmaf(g, x, vz);
  g = G(5); Sp = fmaf(Gp(5), yz, Sp); vy = fmaf(g, z, vy); vz = fmaf(g, y, vz);
  g = G(6); Sp = fmaf(Gp(6), c2, Sp); vx = fmaf(g, 2.0f * x, vx); vy = fmaf(g, -2.0f * y, vy);
  g = G(7); Sp = fmaf(Gp(7), s2, Sp); vx = fmaf(g, 2.0f * y, vx); vy = fmaf(g, 2.0f * x, vy);
  // l = 3
  g = G(8); Sp = fmaf(Gp(8), (5.0f * z2 - 3.0f) * z, Sp); vz = fmaf(g, 15.0f * z2 - 3.0f, vz);
  g = G(9); Sp = fmaf(Gp(9), p31 * x, Sp); vx = fmaf(g, p31, vx); vz = fmaf(g, 10.0f * xz, vz);
  g = G(10); Sp = fmaf(Gp(10), p31 * y, Sp); vy = fmaf(g, p31, vy); vz = fmaf(g, 10.0f * yz, vz);
  g = G(11); Sp = fmaf(Gp(11), z * c2, Sp); vx = fmaf(g, 2.0f * xz, vx); vy = fmaf(g, -2.0f * yz, vy); vz = fmaf(g, c2, vz);
  g = G(12); Sp = fmaf(Gp(12), z * s2, Sp); vx = fmaf(g, 2.0f * yz, vx); vy = fmaf(g, 2.0f * xz, vy); vz = fmaf(g, s2, vz);
  g = G(13); Sp = fmaf(Gp(13), c3, Sp); vx = fmaf(g, 3.0f * c2, vx); vy = fmaf(g, -3.0f * s2, vy);
  g = G(14); Sp = fmaf(Gp(14), s3, Sp); vx = fmaf(g, 3.0f * s2, vx); vy = fmaf(g, 3.0f * c2, vy);
  // l = 4
  g = G(15); Sp = fmaf(Gp(15), (35.0f * z2 - 30.0f) * z2 + 3.0f, Sp); vz = fmaf(g, (140.0f * z2 - 60.0f) * z, vz);
  g = G(16); Sp = fmaf(Gp(16), p41 * x, Sp); vx = fmaf(g, p41, vx); vz = fmaf(g, q41 * x, vz);
  g = G(17); Sp = fmaf(Gp(17), p41 * y, Sp); vy = fmaf(g, p41, vy); vz = fmaf(g, q41 * y, vz);
  g = G(18); Sp = fmaf(Gp(18), p42 * c2, Sp); vx = fmaf(g, 2.0f * p42 * x, vx); vy = fmaf(g, -2.0f * p42 * y, vy); vz = fmaf(g, 14.0f * z * c2, vz);
  g = G(19); Sp = fmaf(Gp(19), p42 * s2, Sp); vx = fmaf(g, 2.0f * p42 * y, vx); vy = fmaf(g, 2.0f * p42 * x, vy); vz = fmaf(g, 14.0f * z * s2, vz);
  g = G(20); Sp = fmaf(Gp(20), z * c3, Sp); vx = fmaf(g, 3.0f * z * c2, vx); vy = fmaf(g, -3.0f * z * s2, vy); vz = fmaf(g, c3, vz);
  g = G(21); Sp = fmaf(Gp(21), z * s3, Sp); vx = fmaf(g, 3.0f * z * s2, vx); vy = fmaf(g, 3.0f * z * c2, vy); vz = fmaf(g, s3, vz);
  g = G(22); Sp = fmaf(Gp(22), c4, Sp); vx = fmaf(g, 4.0f * c3, vx); vy = fmaf(g, -4.0f * s3, vy);
  g = G(23); Sp = fmaf(Gp(23), s4, Sp); vx = fmaf(g, 4.0f * s3, vx); vy = fmaf(g, 4.0f * c3, vy);
}

// cos(pi t) and sin(pi t) for t in [0, 1] (t = r/rc inside the cutoff): with y = 1/2 - t in [-1/2, 1/2],
// cos(pi t) = sin(pi y) = y P(y^2), sin(pi t) = cos(pi y) = Q(y^2).  P, Q: Chebyshev interpolants of
// sin(pi sqrt(w))/sqrt(w) and cos(pi sqrt(w)) on w in [0, 1/4] (degree 4 / 5; truncation error 7e-9 / 2e-10,
// below fp32 rounding).  Replaces sincospif (range reduction not needed here): ~12 instructions for both.
__device__ __forceinline__ float cospi_unit(float t, float& y, float& w) {
  y = 0.5f - t;
  w = y * y;
  float p = fmaf(w, 7.765591228e-02f, -5.982904113e-01f);
  p = fmaf(w, p, 2.550077387e+00f);
  p = fmaf(w, p, -5.167710077e+00f);
  p = fmaf(w, p, 3.141592640e+00f);
  return y * p;
}
__device__ __forceinline__ float sinpi_unit_from_w(float w) {
  float q = fmaf(w, -2.439593201e-02f, 2.349370685e-01f);
  q = fmaf(w, q, -1.335211949e+00f);
  q = fmaf(w, q, 4.058709155e+00f);
  q = fmaf(w, q, -4.934802137e+00f);
  return fmaf(w, q, 9.999999998e-01f);
}

// cutoff function f_c and Chebyshev polynomials T_0..T_{K-1} at distance r (r < rc)
template <int K>
__device__ __forceinline__ void cheb_T_fwd(float r, float inv_rc, float& fc, float T[K]) {
  float t = r * inv_rc, y, w;
  fc = fmaf(0.5f, cospi_unit(t, y, w), 0.5f);
  float u = t - 1.0f;
  float x = fmaf(2.0f * u, u, -1.0f);
  T[0] = 1.0f;
  if (K > 1) T[1] = x;
  float x2 = 2.0f * x;
#pragma unroll
  for (int k = 2; k < K; ++k) T[k] = fmaf(x2, T[k - 1], -T[k - 2]);
}
// the same plus derivatives: dfc = f_c'(r), x, dx = dx/dr
template <int K>
__device__ __forceinline__ void cheb_T(float r, float inv_rc, float& fc, float& dfc, float& x,
                                       float& dx, float T[K]) {
  float t = r * inv_rc, y, w;
  fc = fmaf(0.5f, cospi_unit(t, y, w), 0.5f);
  dfc = -0.5f * NEPZBL_PI_F * inv_rc * sinpi_unit_from_w(w);
  float u = t - 1.0f;
  x = fmaf(2.0f * u, u, -1.0f);
  dx = 4.0f * u * inv_rc;
  T[0] = 1.0f;
  if (K > 1) T[1] = x;
  float x2 = 2.0f * x;
#pragma unroll
  for (int k = 2; k < K; ++k) T[k] = fmaf(x2, T[k - 1], -T[k - 2]);
}
// Chebyshev polynomials of the second kind U_0..U_{K-2}  (T_k' = k U_{k-1})
template <int K>
__device__ __forceinline__ void cheb_U(float x, float U[K]) {
  U[0] = 1.0f;
  float x2 = 2.0f * x;
  if (K > 1) U[1] = x2;
#pragma unroll
  for (int k = 2; k < K; ++k) U[k] = fmaf(x2, U[k - 1], -U[k - 2]);
}

// One entry of adisp (written by k_radial, streamed by the angular kernels).  One atom type: {rhat, r} -- the
// consumers need nothing else (the back-pass takes 1/r with one MUFU), and all four components of the loaded quad are
// live: with {dx, dy, dz, unused} ptxas reused the dead .w register of a request still in flight as a temporary,
// and that write waited for the load (ncu: long-scoreboard stall in the middle of the forward iteration).
// Several types: {dx, dy, dz, neighbour type}.
template <int NT, bool RINV>
__device__ __forceinline__ void unpack_disp(const float4& d, float& ux, float& uy, float& uz, float& r, float& rinv) {
  if (NT == 1) {
    ux = d.x; uy = d.y; uz = d.z; r = d.w;
    rinv = RINV ? rcp_fast(r) : 0.0f;
  } else {
    const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
    rinv = rsqrt_fast(r2);
    r = r2 * rinv;
    ux = d.x * rinv; uy = d.y * rinv; uz = d.z * rinv;
  }
}
// a harmless entry (r = 1) in either format: {rhat = x, r = 1} or {d = x, type 0}
template <int NT>
__device__ __forceinline__ float4 disp_dummy() { return make_float4(1.0f, 0.0f, 0.0f, NT == 1 ? 1.0f : 0.0f); }

// 16-byte asynchronous copy global -> shared (no destination register: any number in flight)
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(tc05::smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}
// request a line into L1 without a destination register: issued two iterations ahead of the load that uses it
// (ptxas places that load, which needs eight registers across the most register-hungry part of the iteration,
// half an iteration before its use: ncu showed the remaining latency as a long-scoreboard stall at the loop end)
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" :: "l"(p)); }

// NT > 1: the folded angular coefficients of every ordered type pair live in shared memory (ct rows, then k * ct rows),
// each row padded to CT_ROW floats so that a channel's coefficients are three aligned LDS.128 instead of nine scalar loads
#define CT_ROW 12
__device__ __forceinline__ void ld_ct_row(const float* __restrict__ s_cta, int row, float c[CT_ROW]) {
#pragma unroll
  for (int v4 = 0; v4 < CT_ROW / 4; ++v4)
    *reinterpret_cast<float4*>(c + 4 * v4) = *reinterpret_cast<const float4*>(s_cta + row * CT_ROW + 4 * v4);
}

__device__ __forceinline__ float tanh_fast(float z) {
  // 1 - 2/(e^{2z}+1): absolute error ~1e-7, enough for the 1e-5 eV energy tolerance.  The two MUFU
  // operations are issued as they are (ex2.approx.ftz, rcp.approx.ftz): __expf / __fdividef wrap them in range
  // fix-ups (FSETP + predicated FMULs for denormal results / huge denominators) that this expression does not need --
  // e underflows to 0 (tanh = -1) or overflows to inf (rcp(inf) = 0, tanh = 1) at the right limits.  5 instructions.
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(z * 2.8853900817779268f));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(e + 1.0f));
  return fmaf(-2.0f, r, 1.0f);
}

// ------------------------------------------------------------------------- S3: radial descriptor
// q_n = sum_j g^R_n(r_ij) for r_ij < rc_radial; also flags atoms with a neighbour inside the ZBL range.
// RADIAL_LANES lanes per atom: lane p owns list entries p, p+4, ...  The gathers are latency-bound
// (ncu: long-scoreboard stalls on the dependent index -> position loads), so every lane issues 4
// independent index loads and 4 independent position gathers per iteration before any arithmetic.
// Which of a lane's entries are inside the cutoff is kept as a bit mask (word w, bit b <-> entry
// p + 4 (32 w + b)) and handed to k_force, which then gathers only those.  The K basis sums are combined over the 4 lanes
// by a fixed-order shuffle tree (deterministic).
// The same pass serves the angular descriptor: the first nn_a entries of the list are the angular list
// (k_nbr).  For those, the displacement vectors of the entries inside rc_angular are compacted in list
// order into adisp[c][s] (c = 0 .. popc(amask[s]) - 1) and their slots into the bit mask amask[w][s] (AW = 1 or 2 64-bit
// words per atom: list capacities up to 128; word 1 exists only when cap_angular > 64 -- a template parameter of every
// kernel that walks the mask, because a run-time second word cost the common case 1-8 % in k_force / the angular kernels).
// k_angular_nn holds 120 accumulators per thread and runs at 2 warps per scheduler, where it cannot
// hide gather latency; this kernel can, so the gathers live here and k_angular_nn streams adisp with
// coalesced loads.
#define RADIAL_LANES 4
#define RADIAL_UNROLL 4
#ifndef RADIAL_BLOCK
// one warp (8 atoms) per block: the grid is ~1.7 waves of resident threads, and the partly filled last wave
// costs one block's duration -- 128-thread blocks: 49.4 us, 64: 48.6, 32: 47.7 (256 / 512: worse)
#define RADIAL_BLOCK 64  // upper bound; the host launches 32 or 64 threads per block (nepzbl_handle::gather_block)
#endif
// STAGE > 0 (stage.cuh, an experiment): the block is one tile of STAGE_TILE atoms whose neighbour ranges are copied
// to shared memory first (1: plain copies, 2: bulk copies); list entries then come from nl_loc (16-bit offsets).
// Two types: capped at 80 registers (ptxas takes 92 otherwise: 57 against 53 us at 128 000 atoms).  One type: no cap --
// 70 registers / 27 warps per SM beat 64 / 31 (2.04 against 2.13 ms at 8.192 M atoms).
template <class MS, bool TRI, int STAGE = 0, int AW = 1>
__global__ void __launch_bounds__(STAGE ? STAGE_TILE * 4 : RADIAL_BLOCK, (MS::NT > 1 && !STAGE) ? 768 / RADIAL_BLOCK : 0)
k_radial(Scalars* sc, const BoxMap* __restrict__ bm, int n, int npad,
         const int4* __restrict__ xyzt, const int* __restrict__ nn_r, const int* __restrict__ nl_r,
         const __grid_constant__ ModelTables<MS> mt, float* __restrict__ q_radial,
         unsigned* __restrict__ rmask, unsigned* __restrict__ tmask, int mask_words, int* __restrict__ zbl_list,
         const int* __restrict__ nn_a, unsigned long long* __restrict__ amask, float4* __restrict__ adisp,
         const unsigned long long* __restrict__ shellq, const TileDesc* __restrict__ tiles,
         const unsigned short* __restrict__ nl_loc) {
  extern __shared__ __align__(16) unsigned char s_stage[];  // STAGE: [TileDesc | mbarrier | int4 x STAGE_CAP]
  bool staged = false;
  const int4* s_xyzt = nullptr;
  if (STAGE) {
    TileDesc* sd = reinterpret_cast<TileDesc*>(s_stage);
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(s_stage + sizeof(TileDesc));
    int4* sx = reinterpret_cast<int4*>(s_stage + ((sizeof(TileDesc) + 8 + 15) / 16) * 16);
    stage_tile<STAGE == 2 ? 2 : 1>(tiles + blockIdx.x, xyzt, sx, sd, mbar);
    staged = sd->nranges >= 0;
    s_xyzt = sx;
  }
  const int gt = blockIdx.x * blockDim.x + threadIdx.x;
  const int s = gt / RADIAL_LANES, sub = gt % RADIAL_LANES;
  const bool valid = s < n;
  const int sc_ = valid ? s : 0;
  const int4 me = xyzt[sc_];
  float hm[9];  // fixed-point difference -> Cartesian displacement (only the diagonal is live for orthogonal boxes)
#pragma unroll
  for (int k = 0; k < 9; ++k) hm[k] = (TRI || k % 4 == 0) ? bm->hm[k] : 0.0f;
  // basis sums per NEIGHBOUR type: q_n = sum_tj sum_k ct^{ti tj}_nk acc[tj][k]
  float acc[MS::NT][MS::KR];
#pragma unroll
  for (int t = 0; t < MS::NT; ++t)
#pragma unroll
    for (int k = 0; k < MS::KR; ++k) acc[t][k] = 0.0f;
  bool close = false;
  int cnt = valid ? nn_r[sc_] : 0;
  const int cnt_a = valid ? nn_a[sc_] : 0;
  {
    // the skin shell is ordered by the distance at the build; with the two largest displacements adding up to D
    // only its entries inside rc + D can have come inside the cutoff (k_nbr, Scalars::disp_sum)
    const unsigned long long sq = valid ? shellq[sc_] : 0ull;
    const int total = (int)(sq >> 56);
    if (total < 255) {  // 255 = saturated count: walk everything
      const int m = min(8, (int)ceilf(sc->disp_sum * mt.inv_shell_w));
      const int reach = m > 0 ? (int)((sq >> (8 * (m - 1))) & 0xFFull) : 0;
      cnt -= total - reach;
    }
  }
  const int* lp = nl_r + nl_at(sub, sc_, npad);  // rows sub, sub + 4, ...: lstride apart
  const unsigned short* lp16 = STAGE ? nl_loc + (size_t)sub * npad + sc_ : nullptr;
  const size_t lstride = (size_t)RADIAL_LANES * npad;
  unsigned mword = 0u;
  unsigned tword = 0u;  // NT > 1: the types of the in-cutoff entries, same bit positions as mword (k_force reads both)
  int bit = 0, word = 0;
  unsigned alo = 0u, ahi = 0u, blo = 0u, bhi = 0u;  // this lane's part of amask (entries 0..63 and, AW = 2, 64..127)
  int abase = 0;                // angular entries of this atom compacted so far
  const unsigned below = (1u << sub) - 1u;
  const int gshift = threadIdx.x & 28;
  // warp-uniform trip count (entries past a lane's own count are guarded), so that the ballots below
  // are taken by all 32 lanes
  const int cnt_max = __reduce_max_sync(0xffffffffu, cnt);
  // the list entries of a round are loaded one round ahead (jn): a round waits for ONE memory latency (the position
  // gathers), not two in a row (23 % of the stall samples sat on the entry -> position dependency, ncu source page)
  int jn[RADIAL_UNROLL];
  if (!(STAGE && staged)) {
#pragma unroll
    for (int u = 0; u < RADIAL_UNROLL; ++u)
      jn[u] = (sub + RADIAL_LANES * u < cnt) ? lp[(size_t)u * lstride] : sc_;
    lp += (size_t)RADIAL_UNROLL * lstride;
  }
  for (int t = sub; t - sub < cnt_max; t += RADIAL_LANES * RADIAL_UNROLL) {
    int j[RADIAL_UNROLL];
    int4 o[RADIAL_UNROLL];
    if (STAGE && staged) {
#pragma unroll
      for (int u = 0; u < RADIAL_UNROLL; ++u)
        j[u] = (t + RADIAL_LANES * u < cnt) ? (int)lp16[(size_t)u * lstride] : 0;
      lp16 += (size_t)RADIAL_UNROLL * lstride;
#pragma unroll
      for (int u = 0; u < RADIAL_UNROLL; ++u) o[u] = s_xyzt[j[u]];
    } else {
#pragma unroll
      for (int u = 0; u < RADIAL_UNROLL; ++u) {
        j[u] = jn[u];
        NZ_CHECK((unsigned)j[u] < (unsigned)n, "k_radial: list entry outside [0, n)");
        o[u] = xyzt[j[u]];
      }
      const int tn = t + RADIAL_LANES * RADIAL_UNROLL;
#pragma unroll
      for (int u = 0; u < RADIAL_UNROLL; ++u)
        jn[u] = (tn + RADIAL_LANES * u < cnt) ? lp[(size_t)u * lstride] : sc_;
      lp += (size_t)RADIAL_UNROLL * lstride;
    }
    const bool ang_round = __any_sync(0xffffffffu, t - sub < cnt_a);  // any lane still in its angular prefix?
#pragma unroll
    for (int u = 0; u < RADIAL_UNROLL; ++u) {
      const int e = t + RADIAL_LANES * u;
      float dx, dy, dz;
      fixed_disp<TRI>(hm, o[u].x - me.x, o[u].y - me.y, o[u].z - me.z, dx, dy, dz);
      float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
      if (ang_round) {
        const bool pa = e < cnt_a && r2 < mt.rcA2;
        const unsigned g = (__ballot_sync(0xffffffffu, pa) >> gshift) & 0xFu;
        if (pa) {
          NZ_CHECK(abase + __popc(g & below) < 64 * AW, "k_radial: compacted angular entry beyond the mask");
          if (MS::NT > 1) {
            adisp[(size_t)(abase + __popc(g & below)) * npad + sc_] = make_float4(dx, dy, dz, __int_as_float(o[u].w));
          } else {  // {rhat, r}, see unpack_disp
            const float ri = rsqrt_fast(r2);
            adisp[(size_t)(abase + __popc(g & below)) * npad + sc_] = make_float4(dx * ri, dy * ri, dz * ri, r2 * ri);
          }
          if (AW == 1) {
            if (e < 32) alo |= 1u << e; else ahi |= 1u << (e - 32);
          } else {
            const unsigned bitv = 1u << (e & 31);
            if (e < 32) alo |= bitv; else if (e < 64) ahi |= bitv; else if (e < 96) blo |= bitv; else bhi |= bitv;
          }
        }
        abase += __popc(g);
      }
      if ((e < cnt) && r2 < mt.rcR2) {
        float r = r2 * rsqrt_fast(r2), fc, T[MS::KR];
        cheb_T_fwd<MS::KR>(r, mt.inv_rcR, fc, T);
#pragma unroll
        for (int t = 0; t < MS::NT; ++t) {
          const float ft = (MS::NT == 1 || o[u].w == t) ? fc : 0.0f;
#pragma unroll
          for (int k = 0; k < MS::KR; ++k) acc[t][k] = fmaf(ft, T[k], acc[t][k]);
        }
        close = close || (r2 < mt.zbl_flag_r2);
        mword |= 1u << (bit + u);
        if (MS::NT > 1) tword |= (unsigned)(o[u].w & 1) << (bit + u);
      }
    }
    bit += RADIAL_UNROLL;
    if (bit == 32) {
      if (valid) rmask[((size_t)word * RADIAL_LANES + sub) * npad + sc_] = mword;
      if (MS::NT > 1 && valid) tmask[((size_t)word * RADIAL_LANES + sub) * npad + sc_] = tword;
      mword = 0u;
      tword = 0u;
      bit = 0;
      ++word;
    }
  }
  if (valid)
    for (; word < mask_words; ++word) {
      rmask[((size_t)word * RADIAL_LANES + sub) * npad + s] = mword;
      if (MS::NT > 1) tmask[((size_t)word * RADIAL_LANES + sub) * npad + s] = tword;
      mword = 0u;
      tword = 0u;
    }
#pragma unroll
  for (int t = 0; t < MS::NT; ++t)
#pragma unroll
    for (int k = 0; k < MS::KR; ++k) {
      acc[t][k] += __shfl_xor_sync(0xffffffffu, acc[t][k], 1);
      acc[t][k] += __shfl_xor_sync(0xffffffffu, acc[t][k], 2);
    }
  unsigned cb = __ballot_sync(0xffffffffu, close);
  alo |= __shfl_xor_sync(0xffffffffu, alo, 1); alo |= __shfl_xor_sync(0xffffffffu, alo, 2);
  ahi |= __shfl_xor_sync(0xffffffffu, ahi, 1); ahi |= __shfl_xor_sync(0xffffffffu, ahi, 2);
  if (AW > 1) {
    blo |= __shfl_xor_sync(0xffffffffu, blo, 1); blo |= __shfl_xor_sync(0xffffffffu, blo, 2);
    bhi |= __shfl_xor_sync(0xffffffffu, bhi, 1); bhi |= __shfl_xor_sync(0xffffffffu, bhi, 2);
  }
  if (!valid) return;
  if (sub == 0) {
    amask[s] = ((unsigned long long)ahi << 32) | alo;
    if (AW > 1) amask[(size_t)npad + s] = ((unsigned long long)bhi << 32) | blo;
  }
  for (int nq = sub; nq < MS::NR; nq += RADIAL_LANES) {
    float q = 0.0f;
#pragma unroll
    for (int t = 0; t < MS::NT; ++t) {
      const int pr = MS::NT == 1 ? 0 : me.w * MS::NT + t;
#pragma unroll
      for (int k = 0; k < MS::KR; ++k) q = fmaf(mt.ctR[pr][nq][k], acc[t][k], q);
    }
    q_radial[(size_t)nq * npad + s] = q;
  }
  if (sub == 0 && ((cb >> (threadIdx.x & 28)) & 0xFu)) {
    const int slot = atomicAdd(&sc->zbl_count, 1);
    NZ_CHECK((unsigned)slot < (unsigned)n, "k_radial: zbl_list slot");
    zbl_list[slot] = s;
  }
}

// ------------------------------------------------------- S4 + S6 + angular partial forces of S7
// One thread per atom, persistent blocks (grid = resident blocks; a block walks tiles of ANG_THREADS
// atoms), network weights staged in shared memory once per block: w0 [neurons][DPAD], b0, w1 [neurons],
// q_scaler [DPAD].  The kernel holds A[n][lm] (120 values) in registers, which caps it at 2 warps per
// scheduler, so it must not wait on memory (ncu: 27 % of the stall samples of the first version sat on
// the index -> position gathers of its three passes over the list):
//   * no gathers here: k_radial leaves the displacement vectors of the in-cutoff angular neighbours,
//     compacted, in adisp[c][s] and their list slots in amask[s]; the forward and backward passes stream
//     them with coalesced loads issued one iteration ahead;
//   * the forward pass takes two neighbours per iteration (two independent Chebyshev / harmonic
//     chains feeding 240 independent FMAs);
//   * the network takes two neurons per iteration (four independent pre-activation chains, two
//     interleaved tanh evaluations).
// One WARP per block (8 blocks per SM at 255 registers).  With 128-thread blocks the partly filled last round of
// the persistent grid went to warps 0 and 1 of every block, i.e. to two of the four schedulers of each SM while the
// other two idled; single-warp blocks spread it over all four: 98.7 us from 108.2 us at 128 000 atoms (64-thread
// blocks: 106.2).  Capping the registers for a ninth / tenth warp spills and is slower (224: 135 us, 200: 146 us).
#define ANG_THREADS 32
// rows of the staged weight table: n_neurons rounded up to even (two neurons per iteration) plus two
// (the software pipeline reads one pair ahead); the padding rows are zero
// (a multiple of 8: the tensor-core variant walks the neurons in tiles of 8)
__host__ __device__ inline int nn_rows(int n_neurons) { return (((n_neurons + 1) & ~1) + 2 + 7) & ~7; }

// ---- tensor-core variant of the network (north_star: "tensor cores only for the per-atom descriptor x W0 layer and
//      only if ncu shows it beats CUDA-core FMA"; measured verdict in DESIGN.md section 5 / profiles/r2_*).
// A warp tile is 32 atoms: Z[32 x NP] = X[32 x KP] W0^T, then Fp[32 x KP] = T[32 x NP] W0 with T = w1 (1 - tanh^2).
// mma.sync m16n8k8 TF32 with the 3-term operand split x = x_hi + x_lo (x_hi w_hi + x_hi w_lo + x_lo w_hi: fp32-grade
// products, fp32 accumulation).  The C fragments of Z are turned into the A fragments of T in place (the neuron index
// of the second product is permuted consistently in A and B), so nothing moves between the two products.
__device__ __forceinline__ unsigned tf32_hi(float x) {
  unsigned r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void tf32_split(float x, unsigned& hi, unsigned& lo) {
  hi = tf32_hi(x);
  lo = tf32_hi(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float c[4], const unsigned a[4], unsigned b0, unsigned b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// c += a * b with the 3-term split; a given as (hi, lo) fragments, b as two fp32 values split here
__device__ __forceinline__ void mma_3xtf32(float c[4], const unsigned ah[4], const unsigned al[4], float b0, float b1) {
  unsigned bh0, bl0, bh1, bl1;
  tf32_split(b0, bh0, bl0);
  tf32_split(b1, bh1, bl1);
  mma_tf32(c, al, bh0, bh1);
  mma_tf32(c, ah, bl0, bl1);
  mma_tf32(c, ah, bh0, bh1);
}
// ---- tcgen05 variant of the network (NN = 2): the Blackwell-native form of the same two products.  A block is FOUR
//      warps = a tile of 128 atoms = the M = 128 rows of one tcgen05.mma; the accumulators live in tensor memory, where
//      row r belongs to thread r (tcgen05.ld 32x32b), so pre-activations and dU/dq arrive in the thread that owns the
//      atom and nothing is shuffled.  Per tile:  every thread stores its scaled descriptor row, split x = hi + lo (tf32
//      + remainder), K-major into shared memory (column D carries the constant 1 against -b0) -> one thread issues
//      Z = X W0^T as hi*hi + hi*lo + lo*hi (kind::tf32, fp32 accumulation in TMEM) and commits to an mbarrier -> every
//      thread reads its 8-neuron chunks of Z, takes tanh, accumulates U and stores T = w1 (1 - h^2) split the same way
//      -> Fp = T W0 in two K halves (neurons 0..31 while the threads are still working on neurons 32..).
//      W0 / W0^T are split once per block.  Layouts and descriptors: tc05.cuh.
struct TcShape {
  int kp;   // K of the first product: D + 1 (bias column) rounded up to 8
  int kn;   // N of the second product: D rounded up to 16 (tcgen05: N % 16 == 0 at M = 128)
};
template <class MS>
__host__ __device__ constexpr TcShape tc_shape() { return TcShape{(MS::D + 1 + 7) / 8 * 8, (MS::D + 15) / 16 * 16}; }
#define TC_NP 64        // neurons padded to the N of the first product (n_neurons <= 64 - 8 for this variant)
#define TC_TMEM_COLS 128  // Z: columns 0..63, Fp: columns 64..64+kn-1
template <class MS>
__host__ __device__ constexpr size_t tc_smem_bytes() {
  // B1 hi/lo [64][kp] + B2 hi/lo [kn][64] + X hi/lo [128][max(kp,32)] + T hi/lo [128][32] + barrier block, 128-byte aligned
  constexpr TcShape t = tc_shape<MS>();
  constexpr int kx = t.kp > 32 ? t.kp : 32;
  return 128 + 4 * (size_t)(2 * TC_NP * t.kp + 2 * t.kn * TC_NP + 2 * 128 * kx + 2 * 128 * 32) + 64;
}

// NN: 0 = network on the CUDA cores (FFMA, weights broadcast from shared memory), 1 = mma.sync 3xTF32, 2 = tcgen05
template <class MS, int NN = 0, int AW = 1>
__global__ void __launch_bounds__(NN == 2 ? 128 : ANG_THREADS, NN == 2 ? 2 : 8)
k_angular_nn(int n, int npad, const int4* __restrict__ xyzt,
             const unsigned long long* __restrict__ amask, const float4* __restrict__ adisp,
             const __grid_constant__ ModelTables<MS> mt, const float* __restrict__ nnw,
             const float* __restrict__ q_radial, float* __restrict__ u_site,
             AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out,
             const DenseArgs da) {
  constexpr int NA = MS::NA, KA = MS::KA, NR = MS::NR, KR = MS::KR, D = MS::D, DPAD = MS::DPAD;
  constexpr bool MMA = NN == 1;
  constexpr bool TC = NN == 2;
  constexpr int T_ = TC ? 128 : ANG_THREADS;
  extern __shared__ __align__(16) float smem[];
  const int neu2 = (mt.n_neurons + 1) & ~1;
  const int nrow = nn_rows(mt.n_neurons);  // zero rows beyond n_neurons (host: build_nnw)
  float* s_w0 = smem;                  // [nrow][DPAD]
  float* s_b0 = s_w0 + nrow * DPAD;    // [nrow]
  float* s_w1 = s_b0 + nrow;           // [nrow]
  float* s_qs = s_w1 + nrow;           // [DPAD]
  // NT > 1: the folded angular coefficients of every ordered type pair, ct [NT*NT][NA][KA] then k * ct, behind the
  // weights (the neighbour's type picks the table per thread: a shared-memory read, where an indexed read of
  // the constant bank cost 2.4x the one-type kernel time)
  const float* s_cta = s_qs + DPAD;
  constexpr int CT_FLOATS = MS::NT > 1 ? 2 * MS::NT * MS::NT * NA * CT_ROW : 0;
  static_assert(KA <= CT_ROW, "padded coefficient rows hold 12 values");
  // MMA: the warp's X / Fp tile [32][XS] and its 32 site energies behind the tables (XS = 4 mod 32: fragment loads
  // hit 32 distinct banks)
  constexpr int KP = (D + 7) / 8 * 8, XS = KP + 4;
  float* s_x = smem + (nrow * DPAD + 2 * nrow + DPAD + CT_FLOATS);
  float* s_u = s_x + 32 * XS;
  {  // all loads of a thread in flight at once (the table is a multiple of 4 floats, 16-byte aligned)
    const int n4 = (nrow * DPAD + 2 * nrow + DPAD + CT_FLOATS) / 4;
    const float4* src = reinterpret_cast<const float4*>(nnw);
    float4* dst = reinterpret_cast<float4*>(smem);
    for (int t = threadIdx.x; t < n4; t += 4 * T_) {
      float4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) if (t + u * T_ < n4) v[u] = src[t + u * T_];
#pragma unroll
      for (int u = 0; u < 4; ++u) if (t + u * T_ < n4) dst[t + u * T_] = v[u];
    }
  }
  __syncthreads();
  // TC: operand tiles behind the tables (128-byte aligned), tensor memory, the mbarrier the MMAs commit to
  constexpr TcShape tcs = tc_shape<MS>();
  constexpr int TKP = tcs.kp, TKN = tcs.kn, TKX = TKP > 32 ? TKP : 32;
  float *tB1h = nullptr, *tB1l = nullptr, *tB2h = nullptr, *tB2l = nullptr, *tXh = nullptr, *tXl = nullptr, *tTh = nullptr, *tTl = nullptr;
  uint32_t tc_mbar = 0, tc_tmem = 0, tc_phase = 0;
  if (TC) {
    const uintptr_t base = (reinterpret_cast<uintptr_t>(smem + (nrow * DPAD + 2 * nrow + DPAD + CT_FLOATS)) + 127) & ~uintptr_t(127);
    tB1h = reinterpret_cast<float*>(base);   // [64 neurons][TKP]   B of Z = X W0^T (column D: -b0)
    tB1l = tB1h + TC_NP * TKP;
    tB2h = tB1l + TC_NP * TKP;               // [TKN components][64 neurons]   B of Fp = T W0
    tB2l = tB2h + TKN * TC_NP;
    tXh = tB2l + TKN * TC_NP;                // [128 atoms][TKX]: X, later the second half of T
    tXl = tXh + 128 * TKX;
    tTh = tXl + 128 * TKX;                   // [128 atoms][32]: first half of T
    tTl = tTh + 128 * 32;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(tTl + 128 * 32);
    uint32_t* tbase = reinterpret_cast<uint32_t*>(bar + 1);
    for (int e = threadIdx.x; e < TC_NP * TKP; e += T_) {
      const int m = e / TKP, k = e % TKP;
      const float w = m < nrow ? (k < D ? s_w0[m * DPAD + k] : (k == D ? -s_b0[m] : 0.0f)) : 0.0f;
      float hi, lo;
      tc05::split_tf32(w, hi, lo);
      *reinterpret_cast<float*>(reinterpret_cast<char*>(tB1h) + tc05::tile_off(TC_NP, m, k)) = hi;
      *reinterpret_cast<float*>(reinterpret_cast<char*>(tB1l) + tc05::tile_off(TC_NP, m, k)) = lo;
    }
    for (int e = threadIdx.x; e < TKN * TC_NP; e += T_) {
      const int v = e / TC_NP, m = e % TC_NP;
      const float w = (m < nrow && v < D) ? s_w0[m * DPAD + v] : 0.0f;
      float hi, lo;
      tc05::split_tf32(w, hi, lo);
      *reinterpret_cast<float*>(reinterpret_cast<char*>(tB2h) + tc05::tile_off(TKN, v, m)) = hi;
      *reinterpret_cast<float*>(reinterpret_cast<char*>(tB2l) + tc05::tile_off(TKN, v, m)) = lo;
    }
    tc_mbar = tc05::smem_u32(bar);
    if (threadIdx.x < 32) tc05::tmem_alloc<TC_TMEM_COLS>(tc05::smem_u32(tbase));
    if (threadIdx.x == 0) tc05::mbar_init(tc_mbar, 1);
    tc05::fence_smem_to_async();
    tc05::fence_before_sync();
    __syncthreads();
    tc05::fence_after_sync();
    tc_tmem = *tbase;
  }
  // Work is handed out per WARP (tiles of 32 atoms; nothing below synchronises the block), with warp
  // slot = warp_in_block * gridDim.x + blockIdx.x, so that the partly filled last round (4000 warp tiles
  // over 1184 resident warps at 128 000 atoms) is spread over all SMs instead of landing on the first
  // blocks only (measured: no difference at 128 000 atoms, 108.7 us either way).
  // TC: the four warps of a block take four consecutive warp tiles (the block synchronises around its MMAs, so
  // all of them make the same number of rounds; a warp past the end carries empty sites).
  const int ntiles = (n + 31) / 32;
  const int nslots = gridDim.x * (T_ / 32);

  // The start of a tile is a chain of dependent global loads (mask -> count -> first displacements) that two
  // warps per scheduler cannot hide, so it is issued one tile ahead: the next tile's mask at the start of this
  // tile, its first two displacement vectors before this tile's back-pass.
  const float4 dummy = disp_dummy<MS::NT>();
  int tile = TC ? blockIdx.x * (T_ / 32) + (threadIdx.x >> 5) : (threadIdx.x >> 5) * gridDim.x + blockIdx.x;
  unsigned long long mask_nx = 0ull;
  float4 pre0 = dummy, pre1 = dummy;
  {
    const int s0 = tile * 32 + (threadIdx.x & 31);
    if (tile < ntiles && s0 < n) {
      mask_nx = amask[s0];
      const int c0 = __popcll(mask_nx) + (AW > 1 ? __popcll(amask[(size_t)npad + s0]) : 0);
      pre0 = c0 > 0 ? adisp[s0] : dummy;
      pre1 = c0 > 1 ? adisp[(size_t)npad + s0] : dummy;
    }
  }
  for (; TC ? tile - (int)(threadIdx.x >> 5) < ntiles : tile < ntiles; tile += nslots) {
    const int s = tile * 32 + (threadIdx.x & 31);
    const unsigned long long mask = mask_nx;
    const int s2 = (tile + nslots) * 32 + (threadIdx.x & 31);
    const bool v2 = tile + nslots < ntiles && s2 < n;
    mask_nx = v2 ? amask[s2] : 0ull;
    // the tensor-core variant needs all 32 lanes in the network: a lane beyond the last atom carries an empty site
    // (no neighbours, nothing written); the FFMA variant lets it skip the tile
    const bool live = s < n;
    if (!MMA && !TC && !live) continue;
    const int sl = live ? s : 0;
    const unsigned long long mask_hi = (AW > 1 && live) ? amask[(size_t)npad + s] : 0ull;  // entries 64..
    const int nc = live ? __popcll(mask) + __popcll(mask_hi) : 0;
    const float4* dp = adisp + sl;
    const int ti = MS::NT > 1 ? xyzt[sl].w : 0;  // type of the central atom (selects the c^{ti tj} tables)
    float qr[NR];
#pragma unroll
    for (int nq = 0; nq < NR; ++nq) qr[nq] = q_radial[(size_t)nq * npad + sl];

    // ---- S4 forward: A[n][lm] = sum_j g_n(r_ij) b_lm(rhat_ij), two neighbours per iteration
    float A[NA][24];
#pragma unroll
    for (int nq = 0; nq < NA; ++nq)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[nq][lm] = 0.0f;
    float4 nx0 = pre0, nx1 = pre1;
    for (int c = 0; c < nc; c += 2) {
      const float4 d2[2] = {nx0, nx1};
      if (c + 4 < nc) prefetch_l1(dp + (size_t)(c + 4) * npad);
      if (c + 5 < nc) prefetch_l1(dp + (size_t)(c + 5) * npad);
      nx0 = c + 2 < nc ? dp[(size_t)(c + 2) * npad] : dummy;  // in flight during this iteration
      nx1 = c + 3 < nc ? dp[(size_t)(c + 3) * npad] : dummy;
      float g2[2][NA], b2[2][24];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        float ux, uy, uz, r, rinv;
        unpack_disp<MS::NT, false>(d2[h], ux, uy, uz, r, rinv);
        float fc, T[KA];
        cheb_T_fwd<KA>(r, mt.inv_rcA, fc, T);
        if (h == 1 && c + 1 >= nc) fc = 0.0f;
        eval_blm(ux, uy, uz, b2[h]);
        const int pr = MS::NT > 1 ? ti * MS::NT + __float_as_int(d2[h].w) : 0;  // adisp.w = neighbour type
#pragma unroll
        for (int nq = 0; nq < NA; ++nq) {
          float cr[CT_ROW];
          if (MS::NT > 1) ld_ct_row(s_cta, pr * NA + nq, cr);
          float g = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k)
            g = fmaf(MS::NT > 1 ? cr[k] : mt.ctA[0][nq][k], T[k], g);
          g2[h][nq] = g * fc;
        }
      }
#pragma unroll
      for (int nq = 0; nq < NA; ++nq)
#pragma unroll
        for (int lm = 0; lm < 24; ++lm) A[nq][lm] = fmaf(g2[1][nq], b2[1][lm], fmaf(g2[0][nq], b2[0][lm], A[nq][lm]));
    }

    // ---- descriptor vector (SURVEY 8(c) C order), scaled
    float q[D];
#pragma unroll
    for (int nq = 0; nq < NR; ++nq) q[nq] = qr[nq];
#pragma unroll
    for (int nq = 0; nq < NA; ++nq) {
      float ql[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) ql[lm_to_l(lm) - 1] = fmaf(kClm[lm] * A[nq][lm], A[nq][lm], ql[lm_to_l(lm) - 1]);
#pragma unroll
      for (int l = 0; l < 4; ++l) q[NR + l * NA + nq] = ql[l];
      if (MS::B5) q[MS::B5 ? MS::V5 + nq : 0] = ql[0] * ql[0] * (1.0f / 3.0f);
    }
    float q1u[MS::B5 ? NA : 1];     // unscaled q_{n,l=1}: d q5_n / d q_{n1} = 2/3 q_{n1}
    if (MS::B5) {
#pragma unroll
      for (int nq = 0; nq < NA; ++nq) q1u[nq] = q[NR + nq];
    }
    float dq4[MS::B4 ? NA : 1][5];  // d q4_n / d A[n][3..7]
    if (MS::B4) {
#pragma unroll
      for (int nq = 0; nq < NA; ++nq) {
        float a0 = A[nq][3], a1 = A[nq][4], a2 = A[nq][5], a3 = A[nq][6], a4 = A[nq][7];
        float Szz = a0 * (1.0f / 3.0f), Sxz = a1, Syz = a2, Sxy = 0.5f * a4;
        float Sxx = fmaf(-1.0f / 6.0f, a0, 0.5f * a3), Syy = fmaf(-1.0f / 6.0f, a0, -0.5f * a3);
        float cxx = Syy * Szz - Syz * Syz, cyy = Sxx * Szz - Sxz * Sxz, czz = Sxx * Syy - Sxy * Sxy;
        float cxy = Sxz * Syz - Sxy * Szz, cxz = Sxy * Syz - Syy * Sxz, cyz = Sxy * Sxz - Sxx * Syz;
        float det = Sxx * cxx + Sxy * cxy + Sxz * cxz;
        const float k3 = 3.0f * NEPZBL_C4;
        q[NR + 4 * NA + nq] = k3 * det;
        dq4[nq][0] = k3 * ((czz * (1.0f / 3.0f)) - (cxx + cyy) * (1.0f / 6.0f));
        dq4[nq][1] = k3 * 2.0f * cxz;
        dq4[nq][2] = k3 * 2.0f * cyz;
        dq4[nq][3] = k3 * 0.5f * (cxx - cyy);
        dq4[nq][4] = k3 * cxy;
      }
    }
    if (q_out && live) {
#pragma unroll
      for (int v = 0; v < D; ++v) q_out[(size_t)v * npad + s] = q[v];
    }

    // ---- S6: network forward + gradient, two neurons per iteration
    float Fp[D];
#pragma unroll
    for (int v = 0; v < D; ++v) {
      q[v] *= s_qs[v];
      Fp[v] = 0.0f;
    }
    if (da.dense_list && live) {  // large angular inputs: fp32 sums are not accurate enough, list the atom for the fp64 pass
      float mx = 0.0f, mx4 = 0.0f;
#pragma unroll
      for (int v = NR; v < NR + 4 * NA; ++v) mx = fmaxf(mx, fabsf(q[v]));
#pragma unroll
      for (int v = NR + 4 * NA; v < D; ++v) mx4 = fmaxf(mx4, fabsf(q[v]));
      if (!(mx <= mt.dense_thr) || !(mx4 <= mt.dense_thr4)) da.dense_list[atomicAdd(&da.sc->dense_count, 1)] = s;
    }
    float U = -mt.b1;
    if (TC) {
      // ---- tcgen05 path (see the comment above the kernel).  Row of X: q (scaled), 1 in column D, zeros beyond.
      char* const xh = reinterpret_cast<char*>(tXh), * const xl = reinterpret_cast<char*>(tXl);
#pragma unroll
      for (int v4 = 0; v4 < TKP / 4; ++v4) {
        float4 h4, l4;
        float* hp = &h4.x;
        float* lp = &l4.x;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int v = 4 * v4 + e;
          const float x = v < D ? q[v < D ? v : 0] : (v == D ? 1.0f : 0.0f);
          tc05::split_tf32(x, hp[e], lp[e]);
        }
        *reinterpret_cast<float4*>(xh + tc05::tile_off(128, threadIdx.x, 4 * v4)) = h4;
        *reinterpret_cast<float4*>(xl + tc05::tile_off(128, threadIdx.x, 4 * v4)) = l4;
      }
      tc05::fence_smem_to_async();
      tc05::fence_before_sync();
      __syncthreads();
      if (threadIdx.x == 0) {  // Z[128 x 64] = X[128 x TKP] B1^T, K = 8 per instruction
        tc05::fence_after_sync();
        constexpr uint32_t id1 = tc05::idesc_tf32(128, TC_NP);
#pragma unroll
        for (int ks = 0; ks < TKP / 8; ++ks) {
          const uint32_t ao = ks * 2 * 16 * 128, bo = ks * 2 * 16 * TC_NP;
          const uint64_t ah = tc05::smem_desc(tc05::smem_u32(tXh) + ao, 16 * 128, 128);
          const uint64_t al = tc05::smem_desc(tc05::smem_u32(tXl) + ao, 16 * 128, 128);
          const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB1h) + bo, 16 * TC_NP, 128);
          const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB1l) + bo, 16 * TC_NP, 128);
          tc05::mma_tf32(tc_tmem, al, bh, id1, ks > 0);
          tc05::mma_tf32(tc_tmem, ah, bl, id1, true);
          tc05::mma_tf32(tc_tmem, ah, bh, id1, true);
        }
        tc05::commit(tc_mbar);
      }
      __syncwarp();
      tc05::mbar_wait(tc_mbar, tc_phase);
      tc_phase ^= 1u;
      tc05::fence_after_sync();
      const uint32_t trow = tc_tmem + ((uint32_t)(threadIdx.x & 96) << 16);  // TMEM lane base of this warp: 32 (warp % 4)
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        // neurons 32 half .. : tanh, site energy, T = w1 (1 - h^2) split into the A tile of the second product
        // (half 0 -> its own tile; half 1 -> X's tile, which the first product has finished reading)
        char* const th = reinterpret_cast<char*>(half ? tXh : tTh), * const tl = reinterpret_cast<char*>(half ? tXl : tTl);
        const int m_end = min(nrow, 32 * half + 32);
#pragma unroll 1
        for (int m0 = 32 * half; m0 < m_end; m0 += 8) {
          float z[8];
          tc05::tmem_ld8(trow + m0, z);
          float4 h4[2], l4[2];
          float* hp = &h4[0].x;
          float* lp = &l4[0].x;
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const float hh = tanh_fast(z[e]);
            const float w1 = s_w1[m0 + e];  // zero in the padding rows
            U = fmaf(w1, hh, U);
            tc05::split_tf32(w1 * fmaf(-hh, hh, 1.0f), hp[e], lp[e]);
          }
          const int kk = m0 - 32 * half;
          *reinterpret_cast<float4*>(th + tc05::tile_off(128, threadIdx.x, kk)) = h4[0];
          *reinterpret_cast<float4*>(th + tc05::tile_off(128, threadIdx.x, kk + 4)) = h4[1];
          *reinterpret_cast<float4*>(tl + tc05::tile_off(128, threadIdx.x, kk)) = l4[0];
          *reinterpret_cast<float4*>(tl + tc05::tile_off(128, threadIdx.x, kk + 4)) = l4[1];
        }
        tc05::fence_smem_to_async();
        tc05::fence_before_sync();
        __syncthreads();
        if (threadIdx.x == 0) {  // Fp[128 x TKN] += T[128 x (this half's neurons)] B2^T
          tc05::fence_after_sync();
          constexpr uint32_t id2 = tc05::idesc_tf32(128, TKN);
          const int nks = (m_end - 32 * half) / 8;
#pragma unroll 1
          for (int ks = 0; ks < nks; ++ks) {
            const uint32_t ao = ks * 2 * 16 * 128, bo = (8 * half + 2 * ks) * 16 * TKN;
            const uint64_t ah = tc05::smem_desc(tc05::smem_u32(half ? tXh : tTh) + ao, 16 * 128, 128);
            const uint64_t al = tc05::smem_desc(tc05::smem_u32(half ? tXl : tTl) + ao, 16 * 128, 128);
            const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB2h) + bo, 16 * TKN, 128);
            const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB2l) + bo, 16 * TKN, 128);
            tc05::mma_tf32(tc_tmem + TC_NP, al, bh, id2, half > 0 || ks > 0);
            tc05::mma_tf32(tc_tmem + TC_NP, ah, bl, id2, true);
            tc05::mma_tf32(tc_tmem + TC_NP, ah, bh, id2, true);
          }
          if (half) tc05::commit(tc_mbar);
        }
        __syncwarp();
      }
      tc05::mbar_wait(tc_mbar, tc_phase);
      tc_phase ^= 1u;
      tc05::fence_after_sync();
#pragma unroll
      for (int c = 0; c < (D + 7) / 8 * 8; c += 8) {
        float f[8];
        tc05::tmem_ld8(trow + TC_NP + c, f);
#pragma unroll
        for (int e = 0; e < 8; ++e)
          if (c + e < D) Fp[c + e < D ? c + e : 0] = f[e];
      }
      tc05::fence_before_sync();  // the next tile's products (behind its __syncthreads) overwrite Z and Fp
    } else if (MMA) {
      // ---- tensor-core path: this thread's row of X to shared memory, fragments from there
      const int lane = threadIdx.x & 31, g = lane >> 2, tig = lane & 3;
      __syncwarp();
#pragma unroll
      for (int v4 = 0; v4 < KP / 4; ++v4) {
        float4 t4;
        t4.x = 4 * v4 + 0 < D ? q[4 * v4 + 0 < D ? 4 * v4 + 0 : 0] : 0.0f;
        t4.y = 4 * v4 + 1 < D ? q[4 * v4 + 1 < D ? 4 * v4 + 1 : 0] : 0.0f;
        t4.z = 4 * v4 + 2 < D ? q[4 * v4 + 2 < D ? 4 * v4 + 2 : 0] : 0.0f;
        t4.w = 4 * v4 + 3 < D ? q[4 * v4 + 3 < D ? 4 * v4 + 3 : 0] : 0.0f;
        *reinterpret_cast<float4*>(s_x + lane * XS + 4 * v4) = t4;
      }
      __syncwarp();
      // A fragments of X (hi / lo), both 16-row halves of the tile, all k-steps
      unsigned xh[2][KP / 8][4], xl[2][KP / 8][4];
#pragma unroll
      for (int mtl = 0; mtl < 2; ++mtl)
#pragma unroll
        for (int ks = 0; ks < KP / 8; ++ks) {
          const float* xp = s_x + (16 * mtl + g) * XS + 8 * ks + tig;
          tf32_split(xp[0], xh[mtl][ks][0], xl[mtl][ks][0]);
          tf32_split(xp[8 * XS], xh[mtl][ks][1], xl[mtl][ks][1]);
          tf32_split(xp[4], xh[mtl][ks][2], xl[mtl][ks][2]);
          tf32_split(xp[8 * XS + 4], xh[mtl][ks][3], xl[mtl][ks][3]);
        }
      float fpc[2][KP / 8][4];  // Fp tile in C fragments
#pragma unroll
      for (int mtl = 0; mtl < 2; ++mtl)
#pragma unroll
        for (int nt = 0; nt < KP / 8; ++nt)
#pragma unroll
          for (int e = 0; e < 4; ++e) fpc[mtl][nt][e] = 0.0f;
      float ur[2][2] = {{0.0f, 0.0f}, {0.0f, 0.0f}};  // site-energy parts of rows g, g + 8 of both halves
#pragma unroll 1
      for (int nt = 0; nt < nrow / 8; ++nt) {  // 8 neurons at a time: Z tile -> tanh -> T -> Fp += T W0
        float z[2][4];
        const float bz0 = s_b0[8 * nt + 2 * tig], bz1 = s_b0[8 * nt + 2 * tig + 1];
#pragma unroll
        for (int mtl = 0; mtl < 2; ++mtl) { z[mtl][0] = -bz0; z[mtl][1] = -bz1; z[mtl][2] = -bz0; z[mtl][3] = -bz1; }
#pragma unroll
        for (int ks = 0; ks < KP / 8; ++ks) {  // B[k][n] = W0[neuron 8 nt + n][8 ks + k]
          const float* wp = s_w0 + (8 * nt + g) * DPAD + 8 * ks + tig;
          const float b0v = 8 * ks + tig < DPAD ? wp[0] : 0.0f, b1v = 8 * ks + tig + 4 < DPAD ? wp[4] : 0.0f;
          mma_3xtf32(z[0], xh[0][ks], xl[0][ks], b0v, b1v);
          mma_3xtf32(z[1], xh[1][ks], xl[1][ks], b0v, b1v);
        }
        const float w1a = s_w1[8 * nt + 2 * tig], w1b = s_w1[8 * nt + 2 * tig + 1];
        unsigned th[2][4], tl[2][4];
#pragma unroll
        for (int mtl = 0; mtl < 2; ++mtl) {
          const float h0 = tanh_fast(z[mtl][0]), h1 = tanh_fast(z[mtl][1]), h2 = tanh_fast(z[mtl][2]), h3 = tanh_fast(z[mtl][3]);
          ur[mtl][0] = fmaf(w1b, h1, fmaf(w1a, h0, ur[mtl][0]));
          ur[mtl][1] = fmaf(w1b, h3, fmaf(w1a, h2, ur[mtl][1]));
          // A fragment of T for the second product, neuron order permuted: k' = tig <-> neuron 2 tig, k' = tig + 4 <-> 2 tig + 1
          tf32_split(w1a * fmaf(-h0, h0, 1.0f), th[mtl][0], tl[mtl][0]);
          tf32_split(w1a * fmaf(-h2, h2, 1.0f), th[mtl][1], tl[mtl][1]);
          tf32_split(w1b * fmaf(-h1, h1, 1.0f), th[mtl][2], tl[mtl][2]);
          tf32_split(w1b * fmaf(-h3, h3, 1.0f), th[mtl][3], tl[mtl][3]);
        }
#pragma unroll
        for (int n2 = 0; n2 < KP / 8; ++n2) {  // B[k'][n] = W0[neuron 8 nt + 2 tig (+1)][8 n2 + n]
          const float* wp = s_w0 + (8 * nt + 2 * tig) * DPAD + 8 * n2 + g;
          const float b0v = 8 * n2 + g < DPAD ? wp[0] : 0.0f, b1v = 8 * n2 + g < DPAD ? wp[DPAD] : 0.0f;
          mma_3xtf32(fpc[0][n2], th[0], tl[0], b0v, b1v);
          mma_3xtf32(fpc[1][n2], th[1], tl[1], b0v, b1v);
        }
      }
      // rows complete across the four lanes of a group; results back to the owning threads through shared memory
#pragma unroll
      for (int mtl = 0; mtl < 2; ++mtl)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          float u = ur[mtl][hf];
          u += __shfl_xor_sync(0xffffffffu, u, 1);
          u += __shfl_xor_sync(0xffffffffu, u, 2);
          if (tig == 0) s_u[16 * mtl + 8 * hf + g] = u;
        }
      __syncwarp();
#pragma unroll
      for (int mtl = 0; mtl < 2; ++mtl)
#pragma unroll
        for (int n2 = 0; n2 < KP / 8; ++n2) {
          *reinterpret_cast<float2*>(s_x + (16 * mtl + g) * XS + 8 * n2 + 2 * tig) = make_float2(fpc[mtl][n2][0], fpc[mtl][n2][1]);
          *reinterpret_cast<float2*>(s_x + (16 * mtl + 8 + g) * XS + 8 * n2 + 2 * tig) = make_float2(fpc[mtl][n2][2], fpc[mtl][n2][3]);
        }
      __syncwarp();
      U += s_u[lane];
#pragma unroll
      for (int v4 = 0; v4 < KP / 4; ++v4) {
        const float4 t4 = *reinterpret_cast<const float4*>(s_x + lane * XS + 4 * v4);
        if (4 * v4 + 0 < D) Fp[4 * v4 + 0 < D ? 4 * v4 + 0 : 0] = t4.x;
        if (4 * v4 + 1 < D) Fp[4 * v4 + 1 < D ? 4 * v4 + 1 : 0] = t4.y;
        if (4 * v4 + 2 < D) Fp[4 * v4 + 2 < D ? 4 * v4 + 2 : 0] = t4.z;
        if (4 * v4 + 3 < D) Fp[4 * v4 + 3 < D ? 4 * v4 + 3 : 0] = t4.w;
      }
    } else {
    // software pipeline: the pre-activations of neurons m+2, m+3 are accumulated while the tanh of
    // neurons m, m+1 (two dependent MUFU ops) is in flight; rows neu2, neu2+1 of w0/b0 are zero padding
    auto preact = [&](int m, float& za, float& zb) {
      const float4* wa = reinterpret_cast<const float4*>(s_w0 + m * DPAD);  // broadcast LDS.128
      const float4* wb = wa + DPAD / 4;
      float za0 = -s_b0[m], za1 = 0.0f, zb0 = -s_b0[m + 1], zb1 = 0.0f;
#pragma unroll
      for (int v4 = 0; v4 < DPAD / 4; ++v4) {
        float4 w = wa[v4], x = wb[v4];
        if (4 * v4 + 0 < D) { za0 = fmaf(w.x, q[4 * v4 + 0], za0); zb0 = fmaf(x.x, q[4 * v4 + 0], zb0); }
        if (4 * v4 + 1 < D) { za1 = fmaf(w.y, q[4 * v4 + 1], za1); zb1 = fmaf(x.y, q[4 * v4 + 1], zb1); }
        if (4 * v4 + 2 < D) { za0 = fmaf(w.z, q[4 * v4 + 2], za0); zb0 = fmaf(x.z, q[4 * v4 + 2], zb0); }
        if (4 * v4 + 3 < D) { za1 = fmaf(w.w, q[4 * v4 + 3], za1); zb1 = fmaf(x.w, q[4 * v4 + 3], zb1); }
      }
      za = za0 + za1;
      zb = zb0 + zb1;
    };
    float za, zb;
    preact(0, za, zb);
#pragma unroll 1
    for (int m = 0; m < neu2; m += 2) {
      const float ha = tanh_fast(za), hb = tanh_fast(zb);
      preact(m + 2, za, zb);
      const float4* wa = reinterpret_cast<const float4*>(s_w0 + m * DPAD);
      const float4* wb = wa + DPAD / 4;
      float w1a = s_w1[m], w1b = s_w1[m + 1];
      U = fmaf(w1a, ha, U);
      U = fmaf(w1b, hb, U);
      float ta = w1a * fmaf(-ha, ha, 1.0f), tb = w1b * fmaf(-hb, hb, 1.0f);
#pragma unroll
      for (int v4 = 0; v4 < DPAD / 4; ++v4) {
        float4 w = wa[v4], x = wb[v4];
        if (4 * v4 + 0 < D) Fp[4 * v4 + 0] = fmaf(tb, x.x, fmaf(ta, w.x, Fp[4 * v4 + 0]));
        if (4 * v4 + 1 < D) Fp[4 * v4 + 1] = fmaf(tb, x.y, fmaf(ta, w.y, Fp[4 * v4 + 1]));
        if (4 * v4 + 2 < D) Fp[4 * v4 + 2] = fmaf(tb, x.z, fmaf(ta, w.z, Fp[4 * v4 + 2]));
        if (4 * v4 + 3 < D) Fp[4 * v4 + 3] = fmaf(tb, x.w, fmaf(ta, w.w, Fp[4 * v4 + 3]));
      }
    }
    }
#pragma unroll
    for (int v = 0; v < D; ++v) Fp[v] *= s_qs[v];
    if (live) u_site[s] = U;

    // record for the radial back-pass of k_force: position + Fp[0..NR-1] (32 bytes) or position +
    // d_k = sum_n Fp_n ct_nk (64 bytes), see ModelShape::FPREC
    if (!live) {
      // nothing to record for an empty lane
    } else if (MS::FPREC) {
      const int4 me = xyzt[s];
      float f[5];
#pragma unroll
      for (int nq = 0; nq < 5; ++nq) f[nq] = nq < NR ? Fp[nq < NR ? nq : 0] : 0.0f;
      float4* rp = reinterpret_cast<float4*>(reinterpret_cast<char*>(rec) + (size_t)s * 32);
      rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), f[0]);
      rp[1] = make_float4(f[1], f[2], f[3], f[4]);
    } else {
      // NT > 1: one 64-byte record per PARTNER type t, rec[NT * s + t] = {position, d^(t)_k = sum_n Fp_n ct^{ti t}_nk,
      // own type}: k_force gathers the record of (neighbour j, my type), so the gather costs what it costs for one type
      static_assert(KR <= 12, "AtomRec holds 12 coefficients");
      const int4 me = xyzt[s];
#pragma unroll
      for (int t = 0; t < MS::NT; ++t) {
        const int pr = MS::NT > 1 ? ti * MS::NT + t : 0;
        float d[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) d[k] = 0.0f;
#pragma unroll
        for (int k = 0; k < KR; ++k)
#pragma unroll
          for (int nq = 0; nq < NR; ++nq) d[k] = fmaf(Fp[nq], mt.ctR[pr][nq][k], d[k]);
        float4* rp = reinterpret_cast<float4*>(rec + (size_t)MS::NT * s + t);
        rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), d[0]);
        rp[1] = make_float4(d[1], d[2], d[3], d[4]);
        rp[2] = make_float4(d[5], d[6], d[7], d[8]);
        if (KR > 9 || MS::NT > 1) rp[3] = make_float4(d[9], d[10], d[11], __int_as_float(me.w));
      }
    }

    // ---- E[n][lm] = dU/dA[n][lm] (in place)
#pragma unroll
    for (int nq = 0; nq < NA; ++nq) {
      const float f5 = MS::B5 ? Fp[MS::B5 ? MS::V5 + nq : 0] * (2.0f / 3.0f) * q1u[MS::B5 ? nq : 0] : 0.0f;
#pragma unroll
      for (int lm = 0; lm < 24; ++lm)
        A[nq][lm] *= 2.0f * kClm[lm] * (Fp[NR + (lm_to_l(lm) - 1) * NA + nq] + (lm < 3 ? f5 : 0.0f));
      if (MS::B4) {
#pragma unroll
        for (int m5 = 0; m5 < 5; ++m5) A[nq][3 + m5] = fmaf(Fp[NR + 4 * NA + nq], dq4[nq][m5], A[nq][3 + m5]);
      }
    }

    // ---- angular partial forces dU_i/dr_ij for the in-cutoff entries (k_force skips the others)
    int c = 0;
    float4 nx = pre0;  // this tile's first displacement is still there; the next tile's are requested now
    {
      const int c2 = __popcll(mask_nx) + ((AW > 1 && v2) ? __popcll(amask[(size_t)npad + s2]) : 0);
      pre0 = c2 > 0 ? adisp[v2 ? s2 : 0] : dummy;
      pre1 = c2 > 1 ? adisp[(size_t)npad + (v2 ? s2 : 0)] : dummy;
    }
    auto back_word = [&](unsigned long long mbits, int abase) {
    for (unsigned long long m = mbits; m; m &= m - 1, ++c) {
      const int a = abase + __ffsll((long long)m) - 1;
      float ux, uy, uz, r, rinv;
      unpack_disp<MS::NT, true>(nx, ux, uy, uz, r, rinv);
      const float tjw = nx.w;
      if (c + 3 < nc) prefetch_l1(dp + (size_t)(c + 3) * npad);
      nx = c + 1 < nc ? dp[(size_t)(c + 1) * npad] : dummy;  // in flight during this iteration
      float fc, dfc, x, dxdr, T[KA], Uc[KA];
      cheb_T<KA>(r, mt.inv_rcA, fc, dfc, x, dxdr, T);
      cheb_U<KA>(x, Uc);
      float g[NA], dg[NA];
      const int pr = MS::NT > 1 ? ti * MS::NT + __float_as_int(tjw) : 0;
#pragma unroll
      for (int nq = 0; nq < NA; ++nq) {
        float cr[CT_ROW], kcr[CT_ROW];
        if (MS::NT > 1) {
          ld_ct_row(s_cta, pr * NA + nq, cr);
          ld_ct_row(s_cta, (MS::NT * MS::NT + pr) * NA + nq, kcr);
        }
        float p = 0.0f, dp = 0.0f;
#pragma unroll
        for (int k = 0; k < KA; ++k)
          p = fmaf(MS::NT > 1 ? cr[k] : mt.ctA[0][nq][k], T[k], p);
#pragma unroll
        for (int k = 1; k < KA; ++k)
          dp = fmaf(MS::NT > 1 ? kcr[k] : mt.kctA[0][nq][k], Uc[k - 1], dp);
        g[nq] = fc * p;
        dg[nq] = fmaf(dfc, p, fc * dxdr * dp);
      }
      auto G = [&](int lm) {
        float t = 0.0f;
#pragma unroll
        for (int nq = 0; nq < NA; ++nq) t = fmaf(g[nq], A[nq][lm], t);
        return t;
      };
      auto Gp = [&](int lm) {
        float t = 0.0f;
#pragma unroll
        for (int nq = 0; nq < NA; ++nq) t = fmaf(dg[nq], A[nq][lm], t);
        return t;
      };
      float Sp, vx, vy, vz;
      contract_blm_grad(ux, uy, uz, G, Gp, Sp, vx, vy, vz);
      float uv = ux * vx + uy * vy + uz * vz;
      float px = fmaf(ux, Sp, (vx - ux * uv) * rinv);
      float py = fmaf(uy, Sp, (vy - uy * uv) * rinv);
      float pz = fmaf(uz, Sp, (vz - uz * uv) * rinv);
      pforce[(size_t)a * npad + s] = make_float4(px, py, pz, 0.0f);
    }
    };
    back_word(live ? mask : 0ull, 0);
    if (AW > 1) back_word(mask_hi, 64);
  }
  if (TC) {
    tc05::fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) tc05::tmem_dealloc<TC_TMEM_COLS>(tc_tmem);
  }
}
