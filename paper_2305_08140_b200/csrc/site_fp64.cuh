// site_fp64.cuh -- FP64 re-evaluation of the sites where FP32 descriptors are not accurate enough.
//
// Why: the angular network inputs x_nu = s_nu q_nu carry an fp32 rounding error that
// grows with the descriptor itself (3-body: dx ~ 2 sqrt(s C x) dA, 4-body: dx ~ 3 s C4 |S|^2 dS with dA, dS ~ 4e-7
// the rounding of a 14-term fp32 sum).  On lattice-like sites (|x| < 1 at 300 K) this is 1e-6 and the north-star
// tolerances (1e-5 eV, 1e-4 eV/A) hold with a wide margin; on DISORDERED sites -- the molten core of a cascade
// (P:71 is about exactly these close encounters), a random cluster -- x reaches 10-1000, the error 1e-5 ... 1e-3,
// and whenever a neuron is not saturated the energy / force error exceeds the tolerance (measured: up to 2.7x,
// DESIGN.md section 6; tests/test_gpu_disordered.py::test_fp32_alone_misses_the_tolerance keeps the measurement).
// k_angular_nn therefore lists every atom with an angular input above ModelTables::dense_thr, and this kernel evaluates S4 + S6 + the angular half of S7 for the listed atoms again in
// FP64 from the fp64 master positions (as k_zbl does for the pair term), overwriting u_site, the k_force record
// and the atom's partial forces.  None in a thermal crystal; the core atoms of a cascade.
//
// One WARP per listed atom; the lanes are (neighbour slice, angular channel) pairs (see the kernel); the network runs
// with the neurons / descriptor components spread over the lanes.  All sizes are run-time values (SiteModel), so the one
// kernel serves every model shape.  Reductions across lanes are fixed-order butterflies: deterministic.
// Same mathematics as descriptor.cuh, same factorisations, FP64 throughout.
#pragma once
#include "force.cuh"

struct SiteModel {  // tables are library-owned device arrays of doubles
  int NT, NR, KR, NA, KA, B4, B5, D, n_neurons;
  int fprec;           // 1: 32-byte record {position, Fp[0..4]} (ModelShape::FPREC), 0: 64-byte AtomRec per partner type
  const double* ctA;   // folded angular coefficients [NT*NT][NA][KA]
  const double* ctR;   // folded radial coefficients  [NT*NT][NR][KR]
  const double* qs;    // q_scaler [D]
  const double* w0;    // [n_neurons][D]
  const double* b0;    // [n_neurons]
  const double* w1;    // [n_neurons]
  double b1, rcA;
};

#define SITE64_WARPS 4
#define SITE64_PI 3.14159265358979323846264338327950288

// real harmonic polynomials b_lm of a unit vector and their gradients in free (x, y, z); same list and order as
// eval_blm / contract_blm_grad (descriptor.cuh).  f(lm, b, bx, by, bz) is called for lm = 0..23.
template <class F>
__device__ __forceinline__ void blm_and_grad_f64(double x, double y, double z, F f) {
  const double z2 = z * z, x2 = x * x, y2 = y * y;
  const double c2 = x2 - y2, s2 = 2.0 * x * y;
  const double c3 = x * (x2 - 3.0 * y2), s3 = y * (3.0 * x2 - y2);
  const double c4 = c2 * c2 - s2 * s2, s4 = 2.0 * c2 * s2;
  const double p31 = 5.0 * z2 - 1.0, p41 = (7.0 * z2 - 3.0) * z, p42 = 7.0 * z2 - 1.0, q41 = 21.0 * z2 - 3.0;
  f(0, z, 0.0, 0.0, 1.0);
  f(1, x, 1.0, 0.0, 0.0);
  f(2, y, 0.0, 1.0, 0.0);
  f(3, 3.0 * z2 - 1.0, 0.0, 0.0, 6.0 * z);
  f(4, x * z, z, 0.0, x);
  f(5, y * z, 0.0, z, y);
  f(6, c2, 2.0 * x, -2.0 * y, 0.0);
  f(7, s2, 2.0 * y, 2.0 * x, 0.0);
  f(8, (5.0 * z2 - 3.0) * z, 0.0, 0.0, 15.0 * z2 - 3.0);
  f(9, p31 * x, p31, 0.0, 10.0 * x * z);
  f(10, p31 * y, 0.0, p31, 10.0 * y * z);
  f(11, z * c2, 2.0 * x * z, -2.0 * y * z, c2);
  f(12, z * s2, 2.0 * y * z, 2.0 * x * z, s2);
  f(13, c3, 3.0 * c2, -3.0 * s2, 0.0);
  f(14, s3, 3.0 * s2, 3.0 * c2, 0.0);
  f(15, (35.0 * z2 - 30.0) * z2 + 3.0, 0.0, 0.0, (140.0 * z2 - 60.0) * z);
  f(16, p41 * x, p41, 0.0, q41 * x);
  f(17, p41 * y, 0.0, p41, q41 * y);
  f(18, p42 * c2, 2.0 * p42 * x, -2.0 * p42 * y, 14.0 * z * c2);
  f(19, p42 * s2, 2.0 * p42 * y, 2.0 * p42 * x, 14.0 * z * s2);
  f(20, z * c3, 3.0 * z * c2, -3.0 * z * s2, c3);
  f(21, z * s3, 3.0 * z * s2, 3.0 * z * c2, s3);
  f(22, c4, 4.0 * c3, -4.0 * s3, 0.0);
  f(23, s4, 4.0 * s3, 4.0 * c3, 0.0);
}

// (2l+1)/(4 pi) times the addition-theorem weight of b_lm
__device__ __forceinline__ double clm_f64(int lm) {
  const double w[24] = {1.0, 1.0, 1.0, 0.25, 3.0, 3.0, 0.75, 0.75, 0.25, 0.375, 0.375, 3.75, 3.75, 0.625, 0.625,
                        1.0 / 64.0, 0.625, 0.625, 0.3125, 0.3125, 4.375, 4.375, 35.0 / 64.0, 35.0 / 64.0};
  const int l = lm_to_l(lm);
  return (2.0 * l + 1.0) / (4.0 * SITE64_PI) * w[lm];
}

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// minimum-image displacement of atom jj from atom i in fp64 (master positions, caller order)
__device__ __forceinline__ void disp_f64(const BoxMap* bm, const double* __restrict__ pos, int n, int i, int jj,
                                         double d[3]) {
#pragma unroll
  for (int a = 0; a < 3; ++a) d[a] = pos[(size_t)a * n + jj] - pos[(size_t)a * n + i];
  min_image_f64(bm, d);
}

// Lane map: lane = slice * NA + n for lane < NS * NA, NS = 32 / NA (config model: 6 slices x 5 channels; paper-sized
// model: 2 x 11).  Slice s takes the in-cutoff angular neighbours number s, s + NS, ... of the atom, so a warp works
// on NS neighbours at a time; A[n][lm] is then summed over the slices in slice order on every lane (the same bits
// everywhere), and in the back-pass the per-channel parts of a neighbour's partial force are summed over n inside
// its slice, again in a fixed order.
__global__ void __launch_bounds__(32 * SITE64_WARPS)
k_site_fp64(const Scalars* sc, const BoxMap* __restrict__ bm, const SiteModel sm, const int* __restrict__ dense_list,
            int n, int npad, const int4* __restrict__ xyzt, const int* __restrict__ nl_r,
            const unsigned long long* __restrict__ amask, int aw, const int* __restrict__ perm,
            const double* __restrict__ pos, const float* __restrict__ q_radial, float* __restrict__ u_site,
            AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out) {
  extern __shared__ double sm64[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int NR = sm.NR, NA = sm.NA, KA = sm.KA, KR = sm.KR, D = sm.D, NT = sm.NT;
  const int per_warp = 2 * D + sm.n_neurons + 16;             // doubles per warp (+16: 128 one-byte slot numbers)
  double* xs = sm64 + (size_t)wib * per_warp;                 // network inputs x_nu
  double* Fp = xs + D;                                        // dU/dq_nu
  double* tt = Fp + D;                                        // w1 (1 - h^2) per neuron
  unsigned char* slot = reinterpret_cast<unsigned char*>(tt + sm.n_neurons);  // list slot of in-cutoff neighbour c
  const int total = sc->dense_count;
  const int NS = 32 / NA;                                     // >= 1 (NA <= 32, checked at create)
  const bool own = lane < NS * NA;
  const int ch = own ? lane % NA : 0, slice = own ? lane / NA : 0;
  const double rc = sm.rcA, inv_rc = 1.0 / sm.rcA;
  const double C4 = -45.0 / (8.0 * sqrt(14.0) * SITE64_PI * sqrt(SITE64_PI));
  for (int t = blockIdx.x * SITE64_WARPS + wib; t < total; t += gridDim.x * SITE64_WARPS) {
    const int s = dense_list[t];
    NZ_CHECK((unsigned)s < (unsigned)n, "k_site_fp64: listed atom outside [0, n)");
    const int i = perm[s];
    const int4 me = xyzt[s];
    const int ti = me.w;
    const unsigned long long mask = amask[s];
    const unsigned long long mask_hi = aw > 1 ? amask[(size_t)npad + s] : 0ull;  // entries 64.. (cap_angular > 64)
    const int nc = __popcll(mask) + __popcll(mask_hi);
    if (lane == 0) {
      int c = 0;
      for (unsigned long long m = mask; m; m &= m - 1) slot[c++] = (unsigned char)(__ffsll((long long)m) - 1);
      for (unsigned long long m = mask_hi; m; m &= m - 1) slot[c++] = (unsigned char)(64 + __ffsll((long long)m) - 1);
    }
    __syncwarp();
    const int rounds = (nc + NS - 1) / NS;

    // ---- S4 forward in fp64: this lane's part of A[ch][lm] (its slice of the neighbours)
    double A[24];
#pragma unroll
    for (int lm = 0; lm < 24; ++lm) A[lm] = 0.0;
    for (int rd = 0; rd < rounds; ++rd) {
      const int c = rd * NS + slice;
      if (!own || c >= nc) continue;
      const int j = nl_r[nl_at(slot[c], s, npad)];
      NZ_CHECK((unsigned)j < (unsigned)n, "k_site_fp64: list entry outside [0, n)");
      double d[3];
      disp_f64(bm, pos, n, i, perm[j], d);
      const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      if (!(r < rc)) continue;  // the fp32 pass kept a pair that fp64 puts at the cutoff: it contributes nothing
      const double tr = r * inv_rc, u = tr - 1.0;
      const double fc = 0.5 + 0.5 * cospi(tr);
      const double x = 2.0 * u * u - 1.0;
      const double* ct = sm.ctA + ((size_t)(ti * NT + xyzt[j].w) * NA + ch) * KA;
      double T0 = 1.0, T1 = x, g = ct[0];
      if (KA > 1) g += ct[1] * x;
      for (int k = 2; k < KA; ++k) {
        const double T2 = 2.0 * x * T1 - T0;
        g += ct[k] * T2;
        T0 = T1;
        T1 = T2;
      }
      g *= fc;
      const double ri = 1.0 / r;
      blm_and_grad_f64(d[0] * ri, d[1] * ri, d[2] * ri,
                       [&](int lm, double b, double, double, double) { A[lm] += g * b; });
    }
    __syncwarp();
    // sum over the slices, slice 0 first, on every lane of the channel (fixed order: the same bits in all slices)
#pragma unroll
    for (int lm = 0; lm < 24; ++lm) {
      const double mine = A[lm];
      double tot = 0.0;
      for (int sl = 0; sl < NS; ++sl) tot += __shfl_sync(0xffffffffu, mine, sl * NA + ch);
      A[lm] = own ? tot : 0.0;
    }

    // ---- descriptor: 3-body q_nl, 4-body q_n^222, scaled into xs[]
    double ql[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int lm = 0; lm < 24; ++lm) ql[lm_to_l(lm) - 1] += clm_f64(lm) * A[lm] * A[lm];
    double q4 = 0.0, dq4[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (sm.B4) {
      const double a0 = A[3], a1 = A[4], a2 = A[5], a3 = A[6], a4 = A[7];
      const double Szz = a0 / 3.0, Sxz = a1, Syz = a2, Sxy = 0.5 * a4;
      const double Sxx = -a0 / 6.0 + 0.5 * a3, Syy = -a0 / 6.0 - 0.5 * a3;
      const double cxx = Syy * Szz - Syz * Syz, cyy = Sxx * Szz - Sxz * Sxz, czz = Sxx * Syy - Sxy * Sxy;
      const double cxy = Sxz * Syz - Sxy * Szz, cxz = Sxy * Syz - Syy * Sxz, cyz = Sxy * Sxz - Sxx * Syz;
      const double k3 = 3.0 * C4;
      q4 = k3 * (Sxx * cxx + Sxy * cxy + Sxz * cxz);
      dq4[0] = k3 * (czz / 3.0 - (cxx + cyy) / 6.0);
      dq4[1] = k3 * 2.0 * cxz;
      dq4[2] = k3 * 2.0 * cyz;
      dq4[3] = k3 * 0.5 * (cxx - cyy);
      dq4[4] = k3 * cxy;
    }
    if (own && slice == 0) {
#pragma unroll
      for (int l = 0; l < 4; ++l) xs[NR + l * NA + ch] = ql[l];
      if (sm.B4) xs[NR + 4 * NA + ch] = q4;
      if (sm.B5) xs[NR + (4 + sm.B4) * NA + ch] = ql[0] * ql[0] / 3.0;  // (1,1,1,1) term, C-27
    }
    for (int nq = lane; nq < NR; nq += 32) xs[nq] = (double)q_radial[(size_t)nq * npad + s];
    __syncwarp();
    for (int v = lane; v < D; v += 32) {
      if (q_out) q_out[(size_t)v * npad + s] = (float)xs[v];
      xs[v] *= sm.qs[v];
    }
    __syncwarp();

    // ---- S6 in fp64: neurons over the lanes, then dU/dq components over the lanes (fixed summation orders)
    double U = 0.0;
    for (int mu = lane; mu < sm.n_neurons; mu += 32) {
      const double* w = sm.w0 + (size_t)mu * D;
      double z = -sm.b0[mu];
      for (int v = 0; v < D; ++v) z += w[v] * xs[v];
      const double h = tanh(z);
      U += sm.w1[mu] * h;
      tt[mu] = sm.w1[mu] * (1.0 - h * h);
    }
    U = warp_sum_f64(U) - sm.b1;
    __syncwarp();
    for (int v = lane; v < D; v += 32) {
      double f = 0.0;
      for (int mu = 0; mu < sm.n_neurons; ++mu) f += tt[mu] * sm.w0[(size_t)mu * D + v];
      Fp[v] = f * sm.qs[v];
    }
    __syncwarp();

    // ---- per-atom outputs for k_force: site energy and the radial back-pass record (layouts of descriptor.cuh)
    if (lane == 0) u_site[s] = (float)U;
    if (sm.fprec) {
      float* rp = reinterpret_cast<float*>(reinterpret_cast<char*>(rec) + (size_t)s * 32);
      if (lane < 3) rp[lane] = __int_as_float(lane == 0 ? me.x : (lane == 1 ? me.y : me.z));
      else if (lane < 8) rp[lane] = lane - 3 < NR ? (float)Fp[lane - 3] : 0.0f;
    } else {
      for (int tp = 0; tp < NT; ++tp) {
        float* rp = reinterpret_cast<float*>(rec + (size_t)NT * s + tp);
        if (lane < 3) rp[lane] = __int_as_float(lane == 0 ? me.x : (lane == 1 ? me.y : me.z));
        else if (lane < 15) {
          const int k = lane - 3;
          double dk = 0.0;
          if (k < KR) {
            const double* ct = sm.ctR + (size_t)(ti * NT + tp) * NR * KR;
            for (int nq = 0; nq < NR; ++nq) dk += Fp[nq] * ct[nq * KR + k];
          }
          rp[lane] = (float)dk;
        } else if (lane == 15) rp[15] = __int_as_float(me.w);
      }
    }

    // ---- E[lm] = dU/dA[ch][lm] (in place; the same on every slice of the channel)
    const double f5 = (sm.B5 && own) ? Fp[NR + (4 + sm.B4) * NA + ch] * (2.0 / 3.0) * ql[0] : 0.0;
#pragma unroll
    for (int lm = 0; lm < 24; ++lm)
      A[lm] *= own ? 2.0 * clm_f64(lm) * (Fp[NR + (lm_to_l(lm) - 1) * NA + ch] + (lm < 3 ? f5 : 0.0)) : 0.0;
    if (sm.B4 && own) {
      const double f4 = Fp[NR + 4 * NA + ch];
#pragma unroll
      for (int m5 = 0; m5 < 5; ++m5) A[3 + m5] += f4 * dq4[m5];
    }

    // ---- angular partial forces dU_i/dr_ij for every slot of the mask (k_force reads exactly those): slice s
    //      evaluates neighbour rd * NS + s, every lane its channel's part, summed over the channels in channel order
    for (int rd = 0; rd < rounds; ++rd) {
      const int c = rd * NS + slice;
      const bool act = own && c < nc;
      double Sp = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, ri = 0.0, ux = 0.0, uy = 0.0, uz = 0.0;
      int a = 0;
      if (act) {
        a = slot[c];
        const int j = nl_r[nl_at(a, s, npad)];
        double d[3];
        disp_f64(bm, pos, n, i, perm[j], d);
        const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (r < rc) {
          const double tr = r * inv_rc, u = tr - 1.0;
          const double fc = 0.5 + 0.5 * cospi(tr);
          const double dfc = -0.5 * SITE64_PI * inv_rc * sinpi(tr);
          const double x = 2.0 * u * u - 1.0, dxdr = 4.0 * u * inv_rc;
          const double* ct = sm.ctA + ((size_t)(ti * NT + xyzt[j].w) * NA + ch) * KA;
          // p = sum_k ct_k T_k,  dp = sum_k ct_k k U_{k-1}   (T_k' = k U_{k-1})
          double T0 = 1.0, T1 = x, U0 = 1.0, U1 = 2.0 * x;
          double p = ct[0], dp = 0.0;
          if (KA > 1) { p += ct[1] * x; dp += ct[1]; }
          for (int k = 2; k < KA; ++k) {
            const double T2 = 2.0 * x * T1 - T0;
            p += ct[k] * T2;
            dp += ct[k] * (double)k * U1;
            const double U2 = 2.0 * x * U1 - U0;
            T0 = T1; T1 = T2; U0 = U1; U1 = U2;
          }
          const double g = fc * p;
          const double dg = dfc * p + fc * dxdr * dp;
          ri = 1.0 / r; ux = d[0] * ri; uy = d[1] * ri; uz = d[2] * ri;
          blm_and_grad_f64(ux, uy, uz, [&](int lm, double b, double bx, double by, double bz) {
            const double e = A[lm];
            Sp += dg * e * b;
            vx += g * e * bx;
            vy += g * e * by;
            vz += g * e * bz;
          });
        }
      }
      __syncwarp();
      double tS = 0.0, tx = 0.0, ty = 0.0, tz = 0.0;
      for (int nq = 0; nq < NA; ++nq) {  // channels of this lane's slice, channel 0 first
        const int src = slice * NA + nq;
        tS += __shfl_sync(0xffffffffu, Sp, src);
        tx += __shfl_sync(0xffffffffu, vx, src);
        ty += __shfl_sync(0xffffffffu, vy, src);
        tz += __shfl_sync(0xffffffffu, vz, src);
      }
      if (act && ch == 0) {
        const double uv = ux * tx + uy * ty + uz * tz;
        const double px = ux * tS + (tx - ux * uv) * ri;
        const double py = uy * tS + (ty - uy * uv) * ri;
        const double pz = uz * tS + (tz - uz * uv) * ri;
        pforce[(size_t)a * npad + s] = make_float4((float)px, (float)py, (float)pz, 0.0f);
      }
    }
    __syncwarp();
  }
}
