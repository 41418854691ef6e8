// force.cuh -- S7 (force / virial accumulation, gather form) and S5 (ZBL pair term).
//
// S7:  F_i = sum_j (dU_i/dr_ij - dU_j/dr_ji),  W_i = sum_j r_ij (x) dU_j/dr_ji.
//   radial part:  dU_i/dr_ij = rhat_ij sum_k d_i[k] (f_c T_k)'(r_ij), d_i[k] = sum_n Fp_i[n] ct_nk,
//                 so F_i += rhat_ij sum_k (d_i[k] + d_j[k]) (f_c T_k)'  -- one gather of d_j per pair;
//   angular part: partial forces stored by k_angular_nn; F_i += p[i][a] - p[j][rev[i][a]].
//   Gather form only: every atom sums its own pairs in list order -> no float atomics, bitwise
//   reproducible.
// S5 (Eq. 1-4; switch P:71): evaluated in FP64 from the fp64 master positions, only for
//   atoms flagged by k_radial as having a neighbour inside r_outer (rare: none in a thermal lattice).
#pragma once
#include "descriptor.cuh"

template <class MS, bool VIRIAL>
__global__ void __launch_bounds__(128)
k_force(const BoxMap* __restrict__ bm, int n, int npad, const int4* __restrict__ xyzt,
        const int* __restrict__ nn_r, const int* __restrict__ nl_r, const int* __restrict__ nn_a,
        const int* __restrict__ nl_a, const unsigned char* __restrict__ rev,
        const __grid_constant__ ModelTables<MS> mt, const float4* __restrict__ dk,
        const float4* __restrict__ pforce, const float* __restrict__ u_site,
        const int* __restrict__ perm, double* __restrict__ energy, float* __restrict__ force,
        float* __restrict__ virial) {
  constexpr int KR = MS::KR;
  static_assert(KR <= 12, "d_k record holds 12 floats");
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const int4 me = xyzt[s];
  const float hx = bm->hf[0], hy = bm->hf[1], hz = bm->hf[2];
  float di[12];
  {
    float4 a = dk[3 * (size_t)s], b = dk[3 * (size_t)s + 1], c = dk[3 * (size_t)s + 2];
    di[0] = a.x; di[1] = a.y; di[2] = a.z; di[3] = a.w; di[4] = b.x; di[5] = b.y; di[6] = b.z;
    di[7] = b.w; di[8] = c.x; di[9] = c.y; di[10] = c.z; di[11] = c.w;
  }
  float fx = 0.0f, fy = 0.0f, fz = 0.0f;
  float w[9];
#pragma unroll
  for (int c = 0; c < 9; ++c) w[c] = 0.0f;

  // ---- radial pairs
  const int cnt = nn_r[s];
  int jn = cnt > 0 ? nl_r[s] : 0;
  for (int t = 0; t < cnt; ++t) {
    int j = jn;
    if (t + 1 < cnt) jn = nl_r[(size_t)(t + 1) * npad + s];
    int4 o = xyzt[j];
    float dx = (float)(o.x - me.x) * hx, dy = (float)(o.y - me.y) * hy, dz = (float)(o.z - me.z) * hz;
    float r2 = dx * dx + dy * dy + dz * dz;
    if (r2 < mt.rcR2) {
      float dj[12];
      {
        float4 a = dk[3 * (size_t)j], b = dk[3 * (size_t)j + 1], c = dk[3 * (size_t)j + 2];
        dj[0] = a.x; dj[1] = a.y; dj[2] = a.z; dj[3] = a.w; dj[4] = b.x; dj[5] = b.y; dj[6] = b.z;
        dj[7] = b.w; dj[8] = c.x; dj[9] = c.y; dj[10] = c.z; dj[11] = c.w;
      }
      float r = sqrtf(r2), rinv = 1.0f / r;
      float fc, dfc, x, dxdr, T[KR], Uc[KR];
      cheb_T<KR>(r, mt.inv_rcR, fc, dfc, x, dxdr, T);
      cheb_U<KR>(x, Uc);
      // sum_k d[k] (f_c T_k)' = f_c' sum_k d[k] T_k + f_c x' sum_{k>=1} d[k] k U_{k-1}
      float ai = 0.0f, bi = 0.0f, aj = 0.0f, bj = 0.0f;
#pragma unroll
      for (int k = 0; k < KR; ++k) {
        ai = fmaf(di[k], T[k], ai);
        aj = fmaf(dj[k], T[k], aj);
      }
#pragma unroll
      for (int k = 1; k < KR; ++k) {
        float ku = (float)k * Uc[k - 1];
        bi = fmaf(di[k], ku, bi);
        bj = fmaf(dj[k], ku, bj);
      }
      float e = fc * dxdr;
      float gi = fmaf(dfc, ai, e * bi);  // dU_i/dr along rhat_ij
      float gj = fmaf(dfc, aj, e * bj);  // dU_j/dr along rhat_ji (same scalar form)
      float fs = (gi + gj) * rinv;
      fx = fmaf(fs, dx, fx);
      fy = fmaf(fs, dy, fy);
      fz = fmaf(fs, dz, fz);
      if (VIRIAL) {  // W_i += r_ij (x) dU_j/dr_ji = -(gj / r) r_ij (x) r_ij
        float ws = -gj * rinv;
        float wx = ws * dx, wy = ws * dy, wz = ws * dz;
        w[0] = fmaf(dx, wx, w[0]); w[1] = fmaf(dx, wy, w[1]); w[2] = fmaf(dx, wz, w[2]);
        w[3] = fmaf(dy, wx, w[3]); w[4] = fmaf(dy, wy, w[4]); w[5] = fmaf(dy, wz, w[5]);
        w[6] = fmaf(dz, wx, w[6]); w[7] = fmaf(dz, wy, w[7]); w[8] = fmaf(dz, wz, w[8]);
      }
    }
  }

  // ---- angular pairs: own partial force minus the neighbour's partial force on the same pair
  const int ca = nn_a[s];
  for (int a = 0; a < ca; ++a) {
    int j = nl_a[(size_t)a * npad + s];
    int b = rev[(size_t)a * npad + s];
    float4 pij = pforce[(size_t)a * npad + s];
    float4 pji = pforce[(size_t)b * npad + j];
    fx += pij.x - pji.x;
    fy += pij.y - pji.y;
    fz += pij.z - pji.z;
    if (VIRIAL) {
      int4 o = xyzt[j];
      float dx = (float)(o.x - me.x) * hx, dy = (float)(o.y - me.y) * hy, dz = (float)(o.z - me.z) * hz;
      w[0] = fmaf(dx, pji.x, w[0]); w[1] = fmaf(dx, pji.y, w[1]); w[2] = fmaf(dx, pji.z, w[2]);
      w[3] = fmaf(dy, pji.x, w[3]); w[4] = fmaf(dy, pji.y, w[4]); w[5] = fmaf(dy, pji.z, w[5]);
      w[6] = fmaf(dz, pji.x, w[6]); w[7] = fmaf(dz, pji.y, w[7]); w[8] = fmaf(dz, pji.z, w[8]);
    }
  }

  // ---- results in the caller's atom order
  int i = perm[s];
  if (energy) energy[i] = (double)u_site[s];
  if (force) {
    force[i] = fx;
    force[(size_t)n + i] = fy;
    force[2 * (size_t)n + i] = fz;
  }
  if (VIRIAL) {
#pragma unroll
    for (int c = 0; c < 9; ++c) virial[(size_t)c * n + i] = w[c];
  }
}

struct ZblParams {
  double r_inner, r_outer;
  int n_terms;
  double c[4], d[4];
  double a_num, a_pow, coulomb_k;
  double Z[8];
  float filter_r2;  // fixed-point prefilter radius^2
};

// S5: U_ZBL = K Z_i Z_j / r * phi(r/a) * f_c(r)   (Eq. 2-4), half to each atom (Eq. 1).
// Adds to energy / force / virial of the flagged atoms (each atom is handled by exactly one thread).
__global__ void __launch_bounds__(64)
k_zbl(const Scalars* sc, const BoxMap* __restrict__ bm, const int* __restrict__ zbl_list, int n,
      int npad, const int4* __restrict__ xyzt, const int* __restrict__ nn_r,
      const int* __restrict__ nl_r, const int* __restrict__ perm, const double* __restrict__ pos,
      const ZblParams zp, double* __restrict__ energy, float* __restrict__ force,
      float* __restrict__ virial) {
  const int total = sc->zbl_count;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
    int s = zbl_list[t];
    int i = perm[s];
    const int4 me = xyzt[s];
    double xi = pos[i], yi = pos[(size_t)n + i], zi = pos[2 * (size_t)n + i];
    double e = 0.0, f[3] = {0.0, 0.0, 0.0}, w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    int cnt = nn_r[s];
    for (int k = 0; k < cnt; ++k) {
      int j = nl_r[(size_t)k * npad + s];
      int4 o = xyzt[j];
      float fdx = (float)(o.x - me.x) * bm->hf[0], fdy = (float)(o.y - me.y) * bm->hf[1],
            fdz = (float)(o.z - me.z) * bm->hf[2];
      if (fdx * fdx + fdy * fdy + fdz * fdz >= zp.filter_r2) continue;
      int jj = perm[j];
      double d[3] = {pos[jj] - xi, pos[(size_t)n + jj] - yi, pos[2 * (size_t)n + jj] - zi};
#pragma unroll
      for (int a = 0; a < 3; ++a)
        if (bm->pbc[a]) d[a] -= bm->L[a] * rint(d[a] / bm->L[a]);  // minimum image in fp64
      double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      if (!(r < zp.r_outer)) continue;
      double Zi = zp.Z[me.w], Zj = zp.Z[o.w];
      double a0 = zp.a_num / (pow(Zi, zp.a_pow) + pow(Zj, zp.a_pow));  // Eq. 4
      double x = r / a0, phi = 0.0, dphi = 0.0;
      for (int q = 0; q < zp.n_terms; ++q) {  // Eq. 3
        double ex = zp.c[q] * exp(-zp.d[q] * x);
        phi += ex;
        dphi -= zp.d[q] / a0 * ex;
      }
      double fc = 1.0, dfc = 0.0;  // Tersoff switch
      if (r > zp.r_inner) {
        double wv = 3.14159265358979323846 / (zp.r_outer - zp.r_inner);
        double sn, cs;
        sincos(wv * (r - zp.r_inner), &sn, &cs);
        fc = 0.5 + 0.5 * cs;
        dfc = -0.5 * wv * sn;
      }
      double coul = zp.coulomb_k * Zi * Zj / r;
      double u = coul * phi * fc;                                                  // Eq. 2
      double du = -coul / r * phi * fc + coul * dphi * fc + coul * phi * dfc;
      e += 0.5 * u;  // Eq. 1: half of the pair energy to each atom
      double fs = du / r;  // F_i = dU/dr * rhat_ij (both halves)
      double ws = -0.5 * fs;  // W_i += r_ij (x) dU_j/dr_ji, dU_j/dr_ji = -1/2 U' rhat_ij
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        f[a] += fs * d[a];
#pragma unroll
        for (int b = 0; b < 3; ++b) w[3 * a + b] += ws * d[a] * d[b];
      }
    }
    if (energy) energy[i] += e;
    if (force)
      for (int a = 0; a < 3; ++a) force[(size_t)a * n + i] = (float)((double)force[(size_t)a * n + i] + f[a]);
    if (virial)
      for (int c = 0; c < 9; ++c) virial[(size_t)c * n + i] = (float)((double)virial[(size_t)c * n + i] + w[c]);
  }
}

// descriptor export (parity tests): [D][npad] sorted -> [n][D] caller order
__global__ void k_export_q(int n, int npad, int D, const int* __restrict__ perm,
                           const float* __restrict__ q_sorted, float* __restrict__ out) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int i = perm[s];
  for (int v = 0; v < D; ++v) out[(size_t)i * D + v] = q_sorted[(size_t)v * npad + s];
}
