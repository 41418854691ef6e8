// descriptor_split.cuh -- S4 + S6 + angular half of S7 for LARGE models (the paper's
// own sizes, n_max 15 / 10, l_max 4, 100 neurons).  Same mathematics as k_angular_nn
// (descriptor.cuh); what changes is the work split: A[n][lm] of an 11-channel model is 264 values, too many
// for one thread's registers, so FOUR lanes share an atom (a warp = 8 atoms):
//   * lane p of the quad owns the angular channels n = p, p+4, p+8 (< NA): A[3][24] = 72 accumulators; every
//     lane walks all angular neighbours (the Chebyshev / harmonic evaluation is repeated per lane, the
//     n-contractions -- the bulk of the work -- are split);
//   * the network: lane p takes the neurons m = p, p+4, ...; the full descriptor is gathered with quad
//     shuffles, the four partial dU/dq vectors are summed by a fixed-order xor butterfly (deterministic);
//   * the back-pass is linear in G_lm = sum_n g_n E_nlm, so every lane contracts its own channels down to a
//     partial force vector and only 3 numbers per neighbour cross the quad.
// Weights and the folded angular coefficients sit in shared memory (lanes of a quad read different rows).
#pragma once
#include "descriptor.cuh"

#define SPLIT_LANES 4
#define SPLIT_THREADS 128
// rows of the staged weight table: n_neurons rounded up to a multiple of 8 (two neurons per lane per iteration)
__host__ __device__ inline int nn_rows_split(int n_neurons) { return (n_neurons + 7) & ~7; }
template <class MS>
__host__ __device__ constexpr int split_smem_floats(int nrow) {
  // w0 [nrow][DPAD], b0 [nrow], w1 [nrow], q_scaler [DPAD], ctA [NSUB*4][KA]
  return nrow * MS::DPAD + 2 * nrow + MS::DPAD + ((MS::NA + 3) / 4 * 4) * MS::KA;
}

// A[NSUB][24] is parked in shared memory while the network runs (q[D] + Fp[D] need its registers; without
// this ptxas spilled ~100 registers to local memory): [NSUB * 24][SPLIT_THREADS] floats behind the table
template <class MS>
__host__ __device__ constexpr int split_stash_floats() {
  return (MS::NA + SPLIT_LANES - 1) / SPLIT_LANES * 24 * SPLIT_THREADS;
}

template <class MS>
__global__ void __launch_bounds__(SPLIT_THREADS)
k_angular_nn_split(int n, int npad, const int4* __restrict__ xyzt,
                   const unsigned long long* __restrict__ amask, const float4* __restrict__ adisp,
                   const __grid_constant__ ModelTables<MS> mt, const float* __restrict__ nnw,
                   const float* __restrict__ q_radial, float* __restrict__ u_site,
                   AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out) {
  constexpr int NA = MS::NA, KA = MS::KA, NR = MS::NR, KR = MS::KR, D = MS::D, DPAD = MS::DPAD;
  constexpr int NSUB = (NA + SPLIT_LANES - 1) / SPLIT_LANES;  // channels per lane
  constexpr int NAP = NSUB * SPLIT_LANES;
  extern __shared__ __align__(16) float smem[];
  const int nrow = nn_rows_split(mt.n_neurons);
  float* s_w0 = smem;                // [nrow][DPAD]
  float* s_b0 = s_w0 + nrow * DPAD;  // [nrow]
  float* s_w1 = s_b0 + nrow;         // [nrow]
  float* s_qs = s_w1 + nrow;         // [DPAD]
  float* s_ct = s_qs + DPAD;         // [NAP][KA], rows >= NA zero
  float* s_stash = smem + split_smem_floats<MS>(nrow) + threadIdx.x;  // this thread's column of the A stash
  {  // the host lays the table out in exactly this order (build_nnw_split); its size is a multiple of 4 floats
    const int n4 = split_smem_floats<MS>(nrow) / 4;
    const float4* src = reinterpret_cast<const float4*>(nnw);
    float4* dst = reinterpret_cast<float4*>(smem);
    for (int t = threadIdx.x; t < n4; t += SPLIT_THREADS) dst[t] = src[t];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, sub = lane & 3, qbase = lane & ~3;
  const unsigned qmask = 0xFu << qbase;  // shuffles inside loops whose trip count differs between quads
  const int ntiles = (n + 7) / 8;
  const int nslots = gridDim.x * (SPLIT_THREADS / 32);
  const float4 dummy = make_float4(1.0f, 0.0f, 0.0f, 0.0f);

  for (int tile = (threadIdx.x >> 5) * gridDim.x + blockIdx.x; tile < ntiles; tile += nslots) {
    const int s = tile * 8 + (lane >> 2);
    const bool valid = s < n;            // all 4 lanes of a quad agree; shuffles below stay inside the quad
    const int sc_ = valid ? s : 0;
    const unsigned long long mask = valid ? amask[sc_] : 0ull;
    const int nc = __popcll(mask);
    const float4* dp = adisp + sc_;
    // ---- S4 forward: A[j][lm] = sum_neighbours g_{n_j}(r) b_lm(rhat)
    float A[NSUB][24];
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] = 0.0f;
    {
      // folded coefficients of this lane's channels (loaded again for the back-pass: they must not stay
      // in registers across the network, which needs q[D] + Fp[D] next to A)
      float ct[NSUB][KA];
#pragma unroll
      for (int j = 0; j < NSUB; ++j)
#pragma unroll
        for (int k = 0; k < KA; ++k) ct[j][k] = s_ct[(sub + SPLIT_LANES * j) * KA + k];
      float4 nx = nc > 0 ? dp[0] : dummy;
      for (int c = 0; c < nc; ++c) {
        const float4 d = nx;
        nx = c + 1 < nc ? dp[(size_t)(c + 1) * npad] : dummy;  // in flight during this iteration
        float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
        float rinv = rsqrtf(r2), r = r2 * rinv;
        float fc, T[KA], b[24];
        cheb_T_fwd<KA>(r, mt.inv_rcA, fc, T);
        eval_blm(d.x * rinv, d.y * rinv, d.z * rinv, b);
#pragma unroll
        for (int j = 0; j < NSUB; ++j) {
          float g = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k) g = fmaf(ct[j][k], T[k], g);
          g *= fc;
#pragma unroll
          for (int lm = 0; lm < 24; ++lm) A[j][lm] = fmaf(g, b[lm], A[j][lm]);
        }
      }
    }

    // ---- descriptor: this lane's angular components, then the full scaled vector via quad shuffles
    float qmine[NSUB][4];
    float dq4[MS::B4 ? NSUB : 1][5];
#pragma unroll
    for (int j = 0; j < NSUB; ++j) {
      float ql[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) ql[lm_to_l(lm) - 1] = fmaf(kClm[lm] * A[j][lm], A[j][lm], ql[lm_to_l(lm) - 1]);
#pragma unroll
      for (int l = 0; l < 4; ++l) qmine[j][l] = ql[l];
    }
    float q4mine[MS::B4 ? NSUB : 1];
    if (MS::B4) {
#pragma unroll
      for (int j = 0; j < NSUB; ++j) {
        float a0 = A[j][3], a1 = A[j][4], a2 = A[j][5], a3 = A[j][6], a4 = A[j][7];
        float Szz = a0 * (1.0f / 3.0f), Sxz = a1, Syz = a2, Sxy = 0.5f * a4;
        float Sxx = fmaf(-1.0f / 6.0f, a0, 0.5f * a3), Syy = fmaf(-1.0f / 6.0f, a0, -0.5f * a3);
        float cxx = Syy * Szz - Syz * Syz, cyy = Sxx * Szz - Sxz * Sxz, czz = Sxx * Syy - Sxy * Sxy;
        float cxy = Sxz * Syz - Sxy * Szz, cxz = Sxy * Syz - Syy * Sxz, cyz = Sxy * Sxz - Sxx * Syz;
        float det = Sxx * cxx + Sxy * cxy + Sxz * cxz;
        const float k3 = 3.0f * NEPZBL_C4;
        q4mine[j] = k3 * det;
        dq4[j][0] = k3 * ((czz * (1.0f / 3.0f)) - (cxx + cyy) * (1.0f / 6.0f));
        dq4[j][1] = k3 * 2.0f * cxz;
        dq4[j][2] = k3 * 2.0f * cyz;
        dq4[j][3] = k3 * 0.5f * (cxx - cyy);
        dq4[j][4] = k3 * cxy;
      }
    }
    float q[D];
#pragma unroll
    for (int nq = 0; nq < NR; ++nq) q[nq] = q_radial[(size_t)nq * npad + sc_];
#pragma unroll
    for (int nq = 0; nq < NA; ++nq) {  // channel nq lives in lane nq & 3, slot nq >> 2 (both compile-time)
#pragma unroll
      for (int l = 0; l < 4; ++l)
        q[NR + l * NA + nq] = __shfl_sync(0xffffffffu, qmine[nq / SPLIT_LANES][l], qbase + (nq % SPLIT_LANES));
      if (MS::B4)
        q[NR + 4 * NA + nq] = __shfl_sync(0xffffffffu, q4mine[MS::B4 ? nq / SPLIT_LANES : 0], qbase + (nq % SPLIT_LANES));
    }
    if (q_out && valid && sub == 0) {
#pragma unroll
      for (int v = 0; v < D; ++v) q_out[(size_t)v * npad + s] = q[v];
    }

    // park A in shared memory until the network is done
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) s_stash[(j * 24 + lm) * SPLIT_THREADS] = A[j][lm];
    asm volatile("" ::: "memory");

    // ---- S6: lane p evaluates the neurons m = p, p+4, ... (two per iteration); partial U and dU/dq
    float Fp[D];
#pragma unroll
    for (int v = 0; v < D; ++v) {
      q[v] *= s_qs[v];
      Fp[v] = 0.0f;
    }
    float U = 0.0f;
#pragma unroll 1
    for (int m = sub; m < nrow; m += 2 * SPLIT_LANES) {
      const float4* wa = reinterpret_cast<const float4*>(s_w0 + m * DPAD);
      const float4* wb = reinterpret_cast<const float4*>(s_w0 + (m + SPLIT_LANES) * DPAD);
      float za0 = -s_b0[m], za1 = 0.0f, zb0 = -s_b0[m + SPLIT_LANES], zb1 = 0.0f;
#pragma unroll
      for (int v4 = 0; v4 < DPAD / 4; ++v4) {
        float4 w = wa[v4], x = wb[v4];
        if (4 * v4 + 0 < D) { za0 = fmaf(w.x, q[4 * v4 + 0], za0); zb0 = fmaf(x.x, q[4 * v4 + 0], zb0); }
        if (4 * v4 + 1 < D) { za1 = fmaf(w.y, q[4 * v4 + 1], za1); zb1 = fmaf(x.y, q[4 * v4 + 1], zb1); }
        if (4 * v4 + 2 < D) { za0 = fmaf(w.z, q[4 * v4 + 2], za0); zb0 = fmaf(x.z, q[4 * v4 + 2], zb0); }
        if (4 * v4 + 3 < D) { za1 = fmaf(w.w, q[4 * v4 + 3], za1); zb1 = fmaf(x.w, q[4 * v4 + 3], zb1); }
      }
      const float ha = tanh_fast(za0 + za1), hb = tanh_fast(zb0 + zb1);
      const float w1a = s_w1[m], w1b = s_w1[m + SPLIT_LANES];  // zero in the padding rows
      U = fmaf(w1a, ha, U);
      U = fmaf(w1b, hb, U);
      const float ta = w1a * fmaf(-ha, ha, 1.0f), tb = w1b * fmaf(-hb, hb, 1.0f);
#pragma unroll
      for (int v4 = 0; v4 < DPAD / 4; ++v4) {
        float4 w = wa[v4], x = wb[v4];
        if (4 * v4 + 0 < D) Fp[4 * v4 + 0] = fmaf(tb, x.x, fmaf(ta, w.x, Fp[4 * v4 + 0]));
        if (4 * v4 + 1 < D) Fp[4 * v4 + 1] = fmaf(tb, x.y, fmaf(ta, w.y, Fp[4 * v4 + 1]));
        if (4 * v4 + 2 < D) Fp[4 * v4 + 2] = fmaf(tb, x.z, fmaf(ta, w.z, Fp[4 * v4 + 2]));
        if (4 * v4 + 3 < D) Fp[4 * v4 + 3] = fmaf(tb, x.w, fmaf(ta, w.w, Fp[4 * v4 + 3]));
      }
    }
    // quad all-reduce in a fixed order: (lane0 + lane1) + (lane2 + lane3) on every lane
    U += __shfl_xor_sync(0xffffffffu, U, 1);
    U += __shfl_xor_sync(0xffffffffu, U, 2);
    U -= mt.b1;
#pragma unroll
    for (int v = 0; v < D; ++v) {
      float f = Fp[v];
      f += __shfl_xor_sync(0xffffffffu, f, 1);
      f += __shfl_xor_sync(0xffffffffu, f, 2);
      Fp[v] = f * s_qs[v];
    }

    // ---- per-atom outputs (one lane of the quad): site energy and the record for k_force's radial pass
    if (valid && sub == 0) {
      u_site[s] = U;
      const int4 me = xyzt[s];
      if (MS::FPREC) {
        float f[5];
#pragma unroll
        for (int nq = 0; nq < 5; ++nq) f[nq] = nq < NR ? Fp[nq < NR ? nq : 0] : 0.0f;
        float4* rp = reinterpret_cast<float4*>(reinterpret_cast<char*>(rec) + (size_t)s * 32);
        rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), f[0]);
        rp[1] = make_float4(f[1], f[2], f[3], f[4]);
      } else {
        static_assert(KR <= 12, "AtomRec holds 12 coefficients");
        float d[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) d[k] = 0.0f;
#pragma unroll
        for (int k = 0; k < KR; ++k)
#pragma unroll
          for (int nq = 0; nq < NR; ++nq) d[k] = fmaf(Fp[nq], mt.ctR[nq][k], d[k]);
        float4* rp = reinterpret_cast<float4*>(rec + s);
        rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), d[0]);
        rp[1] = make_float4(d[1], d[2], d[3], d[4]);
        rp[2] = make_float4(d[5], d[6], d[7], d[8]);
        if (KR > 9) rp[3] = make_float4(d[9], d[10], d[11], 0.0f);
      }
    }

    asm volatile("" ::: "memory");
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] = s_stash[(j * 24 + lm) * SPLIT_THREADS];

    // ---- E[j][lm] = dU/dA[n_j][lm] (in place): pick this lane's channels out of Fp with compile-time indices
#pragma unroll
    for (int j = 0; j < NSUB; ++j) {
      float fl[4] = {0.0f, 0.0f, 0.0f, 0.0f}, f4 = 0.0f;
#pragma unroll
      for (int p = 0; p < SPLIT_LANES; ++p) {
        const int nq = p + SPLIT_LANES * j;
        if (nq < NA && sub == p) {
#pragma unroll
          for (int l = 0; l < 4; ++l) fl[l] = Fp[NR + l * NA + (nq < NA ? nq : 0)];
          if (MS::B4) f4 = Fp[MS::B4 ? NR + 4 * NA + (nq < NA ? nq : 0) : 0];
        }
      }
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] *= 2.0f * kClm[lm] * fl[lm_to_l(lm) - 1];
      if (MS::B4) {
#pragma unroll
        for (int m5 = 0; m5 < 5; ++m5) A[j][3 + m5] = fmaf(f4, dq4[MS::B4 ? j : 0][m5], A[j][3 + m5]);
      }
    }

    // ---- angular partial forces dU_i/dr_ij: every lane contracts its channels, 3 numbers cross the quad
    {
      const float* ctp = s_ct;
      asm volatile("" : "+l"(ctp));  // a fresh load, not the forward pass's registers
      float ct[NSUB][KA];
#pragma unroll
      for (int j = 0; j < NSUB; ++j)
#pragma unroll
        for (int k = 0; k < KA; ++k) ct[j][k] = ctp[(sub + SPLIT_LANES * j) * KA + k];
      int c = 0;
      float4 nx = nc > 0 ? dp[0] : dummy;
      for (unsigned long long m = mask; m; m &= m - 1, ++c) {
        const int a = __ffsll((long long)m) - 1;
        const float dx = nx.x, dy = nx.y, dz = nx.z;
        nx = c + 1 < nc ? dp[(size_t)(c + 1) * npad] : dummy;
        float r2 = dx * dx + dy * dy + dz * dz;
        float rinv = rsqrtf(r2), r = r2 * rinv;
        float fc, dfc, x, dxdr, T[KA], Uc[KA];
        cheb_T<KA>(r, mt.inv_rcA, fc, dfc, x, dxdr, T);
        cheb_U<KA>(x, Uc);
        float kU[KA];
        kU[0] = 0.0f;
#pragma unroll
        for (int k = 1; k < KA; ++k) kU[k] = (float)k * Uc[k - 1];  // T_k' = k U_{k-1}
        const float e = fc * dxdr;
        float g[NSUB], dg[NSUB];
#pragma unroll
        for (int j = 0; j < NSUB; ++j) {
          float p = 0.0f, dpk = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k) p = fmaf(ct[j][k], T[k], p);
#pragma unroll
          for (int k = 1; k < KA; ++k) dpk = fmaf(ct[j][k], kU[k], dpk);
          g[j] = fc * p;
          dg[j] = fmaf(dfc, p, e * dpk);
        }
        float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
        auto G = [&](int lm) {
          float t = 0.0f;
#pragma unroll
          for (int j = 0; j < NSUB; ++j) t = fmaf(g[j], A[j][lm], t);
          return t;
        };
        auto Gp = [&](int lm) {
          float t = 0.0f;
#pragma unroll
          for (int j = 0; j < NSUB; ++j) t = fmaf(dg[j], A[j][lm], t);
          return t;
        };
        float Sp, vx, vy, vz;
        contract_blm_grad(ux, uy, uz, G, Gp, Sp, vx, vy, vz);
        float uv = ux * vx + uy * vy + uz * vz;
        float px = fmaf(ux, Sp, (vx - ux * uv) * rinv);
        float py = fmaf(uy, Sp, (vy - uy * uv) * rinv);
        float pz = fmaf(uz, Sp, (vz - uz * uv) * rinv);
        px += __shfl_xor_sync(qmask, px, 1); px += __shfl_xor_sync(qmask, px, 2);
        py += __shfl_xor_sync(qmask, py, 1); py += __shfl_xor_sync(qmask, py, 2);
        pz += __shfl_xor_sync(qmask, pz, 1); pz += __shfl_xor_sync(qmask, pz, 2);
        if (sub == 0) pforce[(size_t)a * npad + s] = make_float4(px, py, pz, 0.0f);
      }
    }
  }
}
