// descriptor_split.cuh -- S4 + S6 + angular half of S7 for LARGE models (the paper's
// own sizes, n_max 15 / 10, l_max 4, 100 neurons).  Same mathematics as k_angular_nn
// (descriptor.cuh); what changes is the work split: A[n][lm] of an 11-channel model is 264 values, too many
// for one thread's registers, so FOUR lanes share an atom (a warp = 8 atoms):
//   * lane p of the quad owns the angular channels n = p, p+4, p+8 (< NA): A[3][24] = 72 accumulators; every
//     lane walks all angular neighbours (the Chebyshev / harmonic evaluation is repeated per lane, the
//     n-contractions -- the bulk of the work -- are split);
//   * the network sees the descriptor in four SLICES, one per lane (SplitLayout): q and dU/dq never leave their
//     lane; only the four pre-activations of a round (reduce-scatter butterfly, fixed order -> deterministic)
//     and the four tanh derivatives cross the quad;
//   * the back-pass is linear in G_lm = sum_n g_n E_nlm, so every lane contracts its own channels down to a
//     partial force vector and only 3 numbers per neighbour cross the quad.
// Weights and the folded angular coefficients sit in shared memory (lanes of a quad read different rows).
#pragma once
#include "descriptor.cuh"

#define SPLIT_LANES 4
#define SPLIT_THREADS 128

// Who holds what.  Lane p of a quad owns the angular channels n = p + 4 j (j < NSUB) and the radial components
// n = RSUB p + i (i < RSUB).  The network sees the descriptor as four SLICES, one per lane, so that neither q nor
// dU/dq ever has to be gathered: slice entry idx of lane p is
//   idx = 4 j + (l - 1)        -> q_{n_j, l}   (3-body, l = 1..4)
//   idx = 4 NSUB + i           -> q_n radial, n = RSUB p + i
//   idx = 4 NSUB + RSUB + j    -> q^222_{n_j}  (4-body, if the model has it)
// and the host permutes the columns of w0 and q_scaler to match (entries beyond NA / NR are zero).
template <class MS>
struct SplitLayout {
  static constexpr int NSUB = (MS::NA + SPLIT_LANES - 1) / SPLIT_LANES;
  static constexpr int RSUB = (MS::NR + SPLIT_LANES - 1) / SPLIT_LANES;
  static constexpr int NAP = NSUB * SPLIT_LANES;
  static constexpr int SL = 4 * NSUB + RSUB + (MS::B4 ? NSUB : 0);
  static constexpr int SLP = (SL + 3) / 4 * 4;  // slice length, padded to float4
  static constexpr int SLS = SLP + 4;           // slice stride: the four slices of a row fall into disjoint banks
  // canonical descriptor index (SURVEY 8(c) C order) of slice entry idx of lane p, or -1
  __host__ __device__ static constexpr int nu(int p, int idx) {
    if (idx < 4 * NSUB) {
      const int n = p + SPLIT_LANES * (idx / 4), l = idx % 4;
      return n < MS::NA ? MS::NR + l * MS::NA + n : -1;
    }
    if (idx < 4 * NSUB + RSUB) {
      const int n = RSUB * p + (idx - 4 * NSUB);
      return n < MS::NR ? n : -1;
    }
    if (MS::B4 && idx < SL) {
      const int n = p + SPLIT_LANES * (idx - 4 * NSUB - RSUB);
      return n < MS::NA ? MS::NR + 4 * MS::NA + n : -1;
    }
    return -1;
  }
  // rows of the weight table: n_neurons rounded up to a multiple of 4 (one neuron per lane per round)
  __host__ __device__ static constexpr int rows(int n_neurons) { return (n_neurons + 3) & ~3; }
  // table (floats): w0 [nrow][4][SLS] | b0 [nrow] | w1 [nrow] | q_scaler [4][SLS] | ctA [NT*NT][NAP][KA] |
  // ctR [NT*NT][4 RSUB][KR]   (leading index of the coefficient tables: ordered type pair ti * NT + tj)
  static constexpr int NPR = MS::NT * MS::NT;
  __host__ __device__ static constexpr int table_floats(int nrow) {
    return nrow * 4 * SLS + 2 * nrow + 4 * SLS + NPR * (NAP * MS::KA + 4 * RSUB * MS::KR);
  }
  // A[NSUB][24] is parked in shared memory while the network runs: [NSUB * 24][SPLIT_THREADS] floats
  __host__ __device__ static constexpr int stash_floats() { return NSUB * 24 * SPLIT_THREADS; }
};

template <class MS, int AW = 1>
__global__ void __launch_bounds__(SPLIT_THREADS, 3)
k_angular_nn_split(int n, int npad, const int4* __restrict__ xyzt,
                   const unsigned long long* __restrict__ amask, const float4* __restrict__ adisp,
                   const __grid_constant__ ModelTables<MS> mt, const float* __restrict__ nnw,
                   const float* __restrict__ q_radial, float* __restrict__ u_site,
                   AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out,
                   const DenseArgs da) {
  using LY = SplitLayout<MS>;
  static_assert(!MS::B5, "the four-lane kernel has no 5-body slice entries yet");
  constexpr int NT = MS::NT;
  constexpr int KA = MS::KA, NR = MS::NR, KR = MS::KR;
  constexpr int NSUB = LY::NSUB, RSUB = LY::RSUB, SLP = LY::SLP, SLS = LY::SLS, NAP = LY::NAP;
  extern __shared__ __align__(16) float smem[];
  const int nrow = LY::rows(mt.n_neurons);
  float* s_w0 = smem;                     // [nrow][4][SLS]
  float* s_b0 = s_w0 + nrow * 4 * SLS;    // [nrow]
  float* s_w1 = s_b0 + nrow;              // [nrow]
  float* s_qs = s_w1 + nrow;              // [4][SLS]
  float* s_ct = s_qs + 4 * SLS;           // [NT*NT][NAP][KA], rows >= NA zero
  float* s_ctr = s_ct + LY::NPR * NAP * KA;  // [NT*NT][4 RSUB][KR], rows >= NR zero
  float* s_stash = smem + LY::table_floats(nrow) + threadIdx.x;  // this thread's column of the A stash
  {  // the host lays the table out in exactly this order (build_nnw); its size is a multiple of 4 floats
    const int n4 = LY::table_floats(nrow) / 4;
    const float4* src = reinterpret_cast<const float4*>(nnw);
    float4* dst = reinterpret_cast<float4*>(smem);
    for (int t = threadIdx.x; t < n4; t += SPLIT_THREADS) dst[t] = src[t];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, sub = lane & 3, qbase = lane & ~3;
  const unsigned qmask = 0xFu << qbase;  // shuffles inside loops whose trip count differs between quads
  const int ntiles = (n + 7) / 8;
  const int nslots = gridDim.x * (SPLIT_THREADS / 32);
  const float4 dummy = disp_dummy<MS::NT>();

  for (int tile = (threadIdx.x >> 5) * gridDim.x + blockIdx.x; tile < ntiles; tile += nslots) {
    const int s = tile * 8 + (lane >> 2);
    const bool valid = s < n;            // all 4 lanes of a quad agree; shuffles below stay inside the quad
    const int sc_ = valid ? s : 0;
    const unsigned long long mask = valid ? amask[sc_] : 0ull;
    const unsigned long long mask_hi = (AW > 1 && valid) ? amask[(size_t)npad + sc_] : 0ull;  // entries 64..
    const int nc = __popcll(mask) + __popcll(mask_hi);
    const float4* dp = adisp + sc_;
    const int ti = NT > 1 ? xyzt[sc_].w : 0;  // central atom's type: selects the c^{ti tj} tables per neighbour
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
        float ux, uy, uz, r, rinv;
        unpack_disp<NT, false>(d, ux, uy, uz, r, rinv);
        float fc, T[KA], b[24];
        cheb_T_fwd<KA>(r, mt.inv_rcA, fc, T);
        eval_blm(ux, uy, uz, b);
        const float* cts = s_ct + (NT > 1 ? (ti * NT + __float_as_int(d.w)) * NAP * KA : 0);  // adisp.w = neighbour type
#pragma unroll
        for (int j = 0; j < NSUB; ++j) {
          float g = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k) g = fmaf(NT > 1 ? cts[(sub + SPLIT_LANES * j) * KA + k] : ct[j][k], T[k], g);
          g *= fc;
#pragma unroll
          for (int lm = 0; lm < 24; ++lm) A[j][lm] = fmaf(g, b[lm], A[j][lm]);
        }
      }
    }

    // ---- descriptor slice of this lane (SplitLayout): 3-body of its channels, its radial components, 4-body
    float q[SLP];
#pragma unroll
    for (int i = 0; i < SLP; ++i) q[i] = 0.0f;
#pragma unroll
    for (int j = 0; j < NSUB; ++j) {
      float ql[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) ql[lm_to_l(lm) - 1] = fmaf(kClm[lm] * A[j][lm], A[j][lm], ql[lm_to_l(lm) - 1]);
#pragma unroll
      for (int l = 0; l < 4; ++l) q[4 * j + l] = ql[l];
    }
    float dq4[MS::B4 ? NSUB : 1][5];
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
        q[MS::B4 ? 4 * NSUB + RSUB + j : 0] = k3 * det;
        dq4[j][0] = k3 * ((czz * (1.0f / 3.0f)) - (cxx + cyy) * (1.0f / 6.0f));
        dq4[j][1] = k3 * 2.0f * cxz;
        dq4[j][2] = k3 * 2.0f * cyz;
        dq4[j][3] = k3 * 0.5f * (cxx - cyy);
        dq4[j][4] = k3 * cxy;
      }
    }
#pragma unroll
    for (int i = 0; i < RSUB; ++i) {
      const int nq = RSUB * sub + i;
      q[4 * NSUB + i] = nq < NR ? q_radial[(size_t)nq * npad + sc_] : 0.0f;
    }
    if (q_out && valid) {  // descriptor export (parity tests), canonical order
#pragma unroll
      for (int i = 0; i < LY::SL; ++i) {
        int nu = -1;
#pragma unroll
        for (int p = 0; p < SPLIT_LANES; ++p)
          if (sub == p) nu = LY::nu(p, i);
        if (nu >= 0) q_out[(size_t)nu * npad + s] = q[i];
      }
    }

    // park A in shared memory until the network is done
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) s_stash[(j * 24 + lm) * SPLIT_THREADS] = A[j][lm];
    asm volatile("" ::: "memory");

    // ---- S6: four neurons per round.  Every lane forms the partial pre-activations of the four neurons over
    //      ITS slice; a two-step butterfly (fixed order) leaves the complete sum of neuron m0 + p on lane p, which
    //      takes the tanh; the four derivatives go round the quad and every lane accumulates dU/dq of its slice.
    float Fp[SLP];
#pragma unroll
    for (int i = 0; i < SLP; ++i) {
      q[i] *= s_qs[sub * SLS + i];
      Fp[i] = 0.0f;
    }
    if (da.dense_list) {  // large angular inputs anywhere in the quad: list the atom for the fp64 pass (site_fp64.cuh)
      float mx = 0.0f, mx4 = 0.0f;
#pragma unroll
      for (int i = 0; i < SLP; ++i) {
        if (i < 4 * NSUB) mx = fmaxf(mx, fabsf(q[i]));
        else if (i >= 4 * NSUB + RSUB) mx4 = fmaxf(mx4, fabsf(q[i]));
      }
      const bool big = !(mx <= mt.dense_thr) || !(mx4 <= mt.dense_thr4);
      const unsigned bq = (__ballot_sync(0xffffffffu, big) >> qbase) & 0xFu;
      if (bq && valid && sub == 0) da.dense_list[atomicAdd(&da.sc->dense_count, 1)] = s;
    }
    float U = 0.0f;
#pragma unroll 1
    for (int m0 = 0; m0 < nrow; m0 += SPLIT_LANES) {
      float4 w[SPLIT_LANES][SLP / 4];
      float z[SPLIT_LANES];
#pragma unroll
      for (int p = 0; p < SPLIT_LANES; ++p) {
        const float4* wp = reinterpret_cast<const float4*>(s_w0 + ((m0 + p) * SPLIT_LANES + sub) * SLS);
        float z0 = 0.0f, z1 = 0.0f;
#pragma unroll
        for (int v4 = 0; v4 < SLP / 4; ++v4) {
          w[p][v4] = wp[v4];
          z0 = fmaf(w[p][v4].x, q[4 * v4 + 0], z0);
          z1 = fmaf(w[p][v4].y, q[4 * v4 + 1], z1);
          z0 = fmaf(w[p][v4].z, q[4 * v4 + 2], z0);
          z1 = fmaf(w[p][v4].w, q[4 * v4 + 3], z1);
        }
        z[p] = z0 + z1;
      }
      const bool b0 = sub & 1, b1 = sub & 2;
      float k01 = b0 ? z[1] : z[0], k23 = b0 ? z[3] : z[2];
      k01 += __shfl_xor_sync(0xffffffffu, b0 ? z[0] : z[1], 1);
      k23 += __shfl_xor_sync(0xffffffffu, b0 ? z[2] : z[3], 1);
      float zm = b1 ? k23 : k01;
      zm += __shfl_xor_sync(0xffffffffu, b1 ? k01 : k23, 2);
      const float h = tanh_fast(zm - s_b0[m0 + sub]);
      const float w1 = s_w1[m0 + sub];  // zero in the padding rows
      U = fmaf(w1, h, U);
      const float t = w1 * fmaf(-h, h, 1.0f);
#pragma unroll
      for (int p = 0; p < SPLIT_LANES; ++p) {
        const float tp = __shfl_sync(0xffffffffu, t, qbase + p);
#pragma unroll
        for (int v4 = 0; v4 < SLP / 4; ++v4) {
          Fp[4 * v4 + 0] = fmaf(tp, w[p][v4].x, Fp[4 * v4 + 0]);
          Fp[4 * v4 + 1] = fmaf(tp, w[p][v4].y, Fp[4 * v4 + 1]);
          Fp[4 * v4 + 2] = fmaf(tp, w[p][v4].z, Fp[4 * v4 + 2]);
          Fp[4 * v4 + 3] = fmaf(tp, w[p][v4].w, Fp[4 * v4 + 3]);
        }
      }
    }
    // site energy: (lane0 + lane1) + (lane2 + lane3) on every lane
    U += __shfl_xor_sync(0xffffffffu, U, 1);
    U += __shfl_xor_sync(0xffffffffu, U, 2);
    U -= mt.b1;
#pragma unroll
    for (int i = 0; i < SLP; ++i) Fp[i] *= s_qs[sub * SLS + i];

    // ---- per-atom outputs: site energy and the record for k_force's radial pass.  The radial dU/dq are spread
    //      over the quad: every lane contracts its RSUB components, a fixed-order butterfly adds the four parts.
    {
      if (valid && sub == 0) u_site[s] = U;
      // one record per PARTNER type tp (NT > 1: d^(tp)_k = sum_n Fp_n ct^{ti tp}_nk, as k_angular_nn writes them)
#pragma unroll
      for (int tp = 0; tp < NT; ++tp) {
        float d[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) d[k] = 0.0f;
        if (MS::FPREC) {  // record holds Fp[0..4] itself: component n sits on lane n / RSUB, entry n % RSUB
#pragma unroll
          for (int nq = 0; nq < 5; ++nq)
            if (nq < NR) d[nq] = __shfl_sync(0xffffffffu, Fp[4 * NSUB + (nq < NR ? nq % RSUB : 0)], qbase + (nq < NR ? nq / RSUB : 0));
        } else {
          static_assert(KR <= 12, "AtomRec holds 12 coefficients");
          const float* ctr = s_ctr + (NT > 1 ? (ti * NT + tp) * 4 * RSUB * KR : 0);
#pragma unroll
          for (int k = 0; k < KR; ++k) {
            float t = 0.0f;
#pragma unroll
            for (int i = 0; i < RSUB; ++i) t = fmaf(Fp[4 * NSUB + i], ctr[(RSUB * sub + i) * KR + k], t);
            t += __shfl_xor_sync(0xffffffffu, t, 1);
            t += __shfl_xor_sync(0xffffffffu, t, 2);
            d[k] = t;
          }
        }
        if (valid && sub == 0) {
          const int4 me = xyzt[s];
          if (MS::FPREC) {
            float4* rp = reinterpret_cast<float4*>(reinterpret_cast<char*>(rec) + (size_t)s * 32);
            rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), d[0]);
            rp[1] = make_float4(d[1], d[2], d[3], d[4]);
          } else {
            float4* rp = reinterpret_cast<float4*>(rec + (size_t)NT * s + tp);
            rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), d[0]);
            rp[1] = make_float4(d[1], d[2], d[3], d[4]);
            rp[2] = make_float4(d[5], d[6], d[7], d[8]);
            if (KR > 9 || NT > 1) rp[3] = make_float4(d[9], d[10], d[11], __int_as_float(me.w));
          }
        }
      }
    }

    asm volatile("" ::: "memory");
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] = s_stash[(j * 24 + lm) * SPLIT_THREADS];

    // ---- E[j][lm] = dU/dA[n_j][lm] (in place): the slice holds exactly this lane's dU/dq
#pragma unroll
    for (int j = 0; j < NSUB; ++j) {
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] *= 2.0f * kClm[lm] * Fp[4 * j + lm_to_l(lm) - 1];
      if (MS::B4) {
#pragma unroll
        for (int m5 = 0; m5 < 5; ++m5)
          A[j][3 + m5] = fmaf(Fp[MS::B4 ? 4 * NSUB + RSUB + j : 0], dq4[MS::B4 ? j : 0][m5], A[j][3 + m5]);
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
#pragma unroll 1
      for (int mw = 0; mw < AW; ++mw)  // AW = 1 unless cap_angular > 64
      for (unsigned long long m = mw ? mask_hi : mask; m; m &= m - 1, ++c) {
        const int a = 64 * mw + __ffsll((long long)m) - 1;
        float ux, uy, uz, r, rinv;
        unpack_disp<NT, true>(nx, ux, uy, uz, r, rinv);
        const float* cts = ctp + (NT > 1 ? (ti * NT + __float_as_int(nx.w)) * NAP * KA : 0);
        nx = c + 1 < nc ? dp[(size_t)(c + 1) * npad] : dummy;
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
          for (int k = 0; k < KA; ++k) p = fmaf(NT > 1 ? cts[(sub + SPLIT_LANES * j) * KA + k] : ct[j][k], T[k], p);
#pragma unroll
          for (int k = 1; k < KA; ++k) dpk = fmaf(NT > 1 ? cts[(sub + SPLIT_LANES * j) * KA + k] : ct[j][k], kU[k], dpk);
          g[j] = fc * p;
          dg[j] = fmaf(dfc, p, e * dpk);
        }
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
