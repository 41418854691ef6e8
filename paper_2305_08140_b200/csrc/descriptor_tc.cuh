// descriptor_tc.cuh -- S4 + S6 + angular half of S7 with the network layer on the Blackwell tensor cores
// (tcgen05.mma, accumulators in tensor memory), software-pipelined so that the tensor-core latency never shows.
//
// Same mathematics and the same per-atom arithmetic as k_angular_nn (descriptor.cuh); what changes:
//   * a block is FOUR warps = a tile of 128 atoms = the M = 128 rows of one tcgen05.mma; row r of every accumulator
//     belongs to thread r (tcgen05.ld 32x32b), so pre-activations and dU/dq arrive in the thread that owns the atom;
//   * the two products  Z = X W0^T  (X = scaled descriptor, column D = 1 against -b0)  and  Fp = T W0
//     (T = w1 (1 - tanh^2 Z)) run as kind::tf32 with the 3-term operand split x = hi + lo (hi*hi + hi*lo + lo*hi,
//     fp32 accumulation): fp32-grade products, parity with the fp64 oracle at the same tolerances as the FFMA kernel;
//   * the A[n][lm] sums of a tile are PARKED IN TENSOR MEMORY between its forward and its backward pass, which lets
//     a block work on two tiles at once: while the tensor core forms Z of tile i+1 the threads run the back-pass of
//     tile i, and while it forms Fp of tile i+1 they run the forward pass of tile i+2.  Per tile the block
//     synchronises twice (operands complete -> one thread issues the MMAs) and waits on two mbarriers whose MMAs
//     were issued a whole pass earlier.
//
//   iteration:  F(nxt)  ->  wait Fp(cur)  ->  store X(nxt)  ->  A(nxt) <-> A(cur) through TMEM  ->  sync, issue Z(nxt)
//               ->  B(cur): Fp from TMEM, records, dU/dA, pair forces
//               ->  wait Z(nxt)  ->  tanh, U(nxt), store T(nxt)  ->  sync, issue Fp(nxt)  ->  cur = nxt
//
// Tensor memory (256 columns per block, two blocks per SM): Z [0, 64), Fp [64, 64 + kn), parked A [128, 248).
// Shared memory: the weight table of k_angular_nn, then (128-byte aligned) B1 hi/lo [64][kp], B2 hi/lo [kn][64],
// X hi/lo [128][max(kp, 32)] (reused for the neurons 32.. of T once Z is complete), T hi/lo [128][32], 2 mbarriers.
#pragma once
#include "descriptor.cuh"

#define TCP_THREADS 128
#define TCP_TMEM_COLS 256
#define TCP_APARK 128  // first TMEM column of the parked A (120 columns)

template <class MS>
__host__ __device__ constexpr size_t tcp_smem_bytes() { return tc_smem_bytes<MS>(); }

// ---- S4 forward: A[n][lm] = sum_j g_n(r_ij) b_lm(rhat_ij) over the nc compacted in-cutoff neighbours (two per
//      iteration, the next two displacement vectors in flight); pre0 / pre1 are the first two, requested earlier
template <class MS>
__device__ __forceinline__ void tcp_forward(float (&A)[MS::NA][24], int nc, const float4* __restrict__ dp, int npad,
                                            float4 pre0, float4 pre1, const ModelTables<MS>& mt,
                                            const float* __restrict__ s_cta, int ti) {
  constexpr int NA = MS::NA, KA = MS::KA;
  const float4 dummy = disp_dummy<MS::NT>();
#pragma unroll
  for (int nq = 0; nq < NA; ++nq)
#pragma unroll
    for (int lm = 0; lm < 24; ++lm) A[nq][lm] = 0.0f;
  float4 nx0 = pre0, nx1 = pre1;
  for (int c = 0; c < nc; c += 2) {
    const float4 d2[2] = {nx0, nx1};
    if (c + 4 < nc) prefetch_l1(dp + (size_t)(c + 4) * npad);
    if (c + 5 < nc) prefetch_l1(dp + (size_t)(c + 5) * npad);
    nx0 = c + 2 < nc ? dp[(size_t)(c + 2) * npad] : dummy;
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
}

// 3-body components of channel nq from A: q_{n,l} = (2l+1)/(4 pi) sum_m C_lm A_nlm^2
template <class MS>
__device__ __forceinline__ void tcp_q3(const float (&A)[MS::NA][24], int nq, float ql[4]) {
  ql[0] = ql[1] = ql[2] = ql[3] = 0.0f;
#pragma unroll
  for (int lm = 0; lm < 24; ++lm) ql[lm_to_l(lm) - 1] = fmaf(kClm[lm] * A[nq][lm], A[nq][lm], ql[lm_to_l(lm) - 1]);
}
// 4-body component q^222_n = 3 C4 det S_n and its derivatives with respect to A[n][3..7]
__device__ __forceinline__ float tcp_q4(const float* __restrict__ a, float dq4[5]) {
  const float a0 = a[3], a1 = a[4], a2 = a[5], a3 = a[6], a4 = a[7];
  const float Szz = a0 * (1.0f / 3.0f), Sxz = a1, Syz = a2, Sxy = 0.5f * a4;
  const float Sxx = fmaf(-1.0f / 6.0f, a0, 0.5f * a3), Syy = fmaf(-1.0f / 6.0f, a0, -0.5f * a3);
  const float cxx = Syy * Szz - Syz * Syz, cyy = Sxx * Szz - Sxz * Sxz, czz = Sxx * Syy - Sxy * Sxy;
  const float cxy = Sxz * Syz - Sxy * Szz, cxz = Sxy * Syz - Syy * Sxz, cyz = Sxy * Sxz - Sxx * Syz;
  const float det = Sxx * cxx + Sxy * cxy + Sxz * cxz;
  const float k3 = 3.0f * NEPZBL_C4;
  dq4[0] = k3 * ((czz * (1.0f / 3.0f)) - (cxx + cyy) * (1.0f / 6.0f));
  dq4[1] = k3 * 2.0f * cxz;
  dq4[2] = k3 * 2.0f * cyz;
  dq4[3] = k3 * 0.5f * (cxx - cyy);
  dq4[4] = k3 * cxy;
  return k3 * det;
}

// ---- angular partial forces dU_i/dr_ij of atom s for the in-cutoff entries of its list (E = dU/dA in place of A);
//      first is the first displacement vector, requested earlier
template <class MS>
__device__ __forceinline__ void tcp_backward(const float (&A)[MS::NA][24], unsigned long long mask, int nc,
                                             const float4* __restrict__ dp, int npad, float4 first,
                                             const ModelTables<MS>& mt, const float* __restrict__ s_cta, int ti,
                                             float4* __restrict__ pf /* pforce + s */) {
  constexpr int NA = MS::NA, KA = MS::KA;
  const float4 dummy = disp_dummy<MS::NT>();
  int c = 0;
  float4 nx = first;
  for (unsigned long long m = mask; m; m &= m - 1, ++c) {
    const int a = __ffsll((long long)m) - 1;
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
      float p = 0.0f, dpk = 0.0f;
#pragma unroll
      for (int k = 0; k < KA; ++k)
        p = fmaf(MS::NT > 1 ? cr[k] : mt.ctA[0][nq][k], T[k], p);
#pragma unroll
      for (int k = 1; k < KA; ++k)
        dpk = fmaf(MS::NT > 1 ? kcr[k] : mt.kctA[0][nq][k], Uc[k - 1], dpk);
      g[nq] = fc * p;
      dg[nq] = fmaf(dfc, p, fc * dxdr * dpk);
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
    const float uv = ux * vx + uy * vy + uz * vz;
    const float px = fmaf(ux, Sp, (vx - ux * uv) * rinv);
    const float py = fmaf(uy, Sp, (vy - uy * uv) * rinv);
    const float pz = fmaf(uz, Sp, (vz - uz * uv) * rinv);
    pf[(size_t)a * npad] = make_float4(px, py, pz, 0.0f);
  }
}

// the record k_force gathers per radial pair (see k_angular_nn): {position, Fp[0..NR-1]} or, per partner type,
// {position, d_k = sum_n Fp_n ct^{ti t}_nk, own type}
template <class MS>
__device__ __forceinline__ void tcp_write_record(const float* __restrict__ Fp, int4 me, int s, int ti,
                                                 const ModelTables<MS>& mt, AtomRec* __restrict__ rec) {
  constexpr int NR = MS::NR, KR = MS::KR;
  if (MS::FPREC) {
    float f[5];
#pragma unroll
    for (int nq = 0; nq < 5; ++nq) f[nq] = nq < NR ? Fp[nq < NR ? nq : 0] : 0.0f;
    float4* rp = reinterpret_cast<float4*>(reinterpret_cast<char*>(rec) + (size_t)s * 32);
    rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), f[0]);
    rp[1] = make_float4(f[1], f[2], f[3], f[4]);
  } else {
    static_assert(KR <= 12, "AtomRec holds 12 coefficients");
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
}

template <class MS>
__global__ void __launch_bounds__(TCP_THREADS, 2)
k_angular_tc(int n, int npad, const int4* __restrict__ xyzt,
             const unsigned long long* __restrict__ amask, const float4* __restrict__ adisp,
             const __grid_constant__ ModelTables<MS> mt, const float* __restrict__ nnw,
             const float* __restrict__ q_radial, float* __restrict__ u_site,
             AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out,
             const DenseArgs da) {
  constexpr int NA = MS::NA, KA = MS::KA, NR = MS::NR, D = MS::D, DPAD = MS::DPAD;
  constexpr int T_ = TCP_THREADS;
  constexpr TcShape tcs = tc_shape<MS>();
  constexpr int KP = tcs.kp, KN = tcs.kn, KX = KP > 32 ? KP : 32;
  static_assert(NA * 24 <= 128 && (NA * 24) % 8 == 0, "parked A: at most 128 TMEM columns, in chunks of 8");
  static_assert(TC_NP + KN <= TCP_APARK, "Z and Fp sit below the parked A");
  extern __shared__ __align__(16) float smem[];
  const int nrow = nn_rows(mt.n_neurons);  // zero rows beyond n_neurons (host: build_nnw); <= 64 here
  float* s_w0 = smem;                  // [nrow][DPAD]
  float* s_b0 = s_w0 + nrow * DPAD;    // [nrow]
  float* s_w1 = s_b0 + nrow;           // [nrow]
  float* s_qs = s_w1 + nrow;           // [DPAD]
  const float* s_cta = s_qs + DPAD;    // NT > 1: folded angular coefficients of every ordered type pair
  constexpr int CT_FLOATS = MS::NT > 1 ? 2 * MS::NT * MS::NT * NA * CT_ROW : 0;
  static_assert(KA <= CT_ROW, "padded coefficient rows hold 12 values");
  const int tab_floats = nrow * DPAD + 2 * nrow + DPAD + CT_FLOATS;
  for (int t = threadIdx.x; t < tab_floats / 4; t += T_)
    cp_async16(reinterpret_cast<float4*>(smem) + t, reinterpret_cast<const float4*>(nnw) + t);
  // operand tiles (layout: tc05.cuh), the two mbarriers, the TMEM base address
  const uintptr_t base = (reinterpret_cast<uintptr_t>(smem + tab_floats) + 127) & ~uintptr_t(127);
  float* const tB1h = reinterpret_cast<float*>(base);  // [64 neurons][KP]      B of Z = X W0^T (column D: -b0)
  float* const tB1l = tB1h + TC_NP * KP;
  float* const tB2h = tB1l + TC_NP * KP;               // [KN components][64]   B of Fp = T W0
  float* const tB2l = tB2h + KN * TC_NP;
  float* const tXh = tB2l + KN * TC_NP;                // [128][KX]: X, later the neurons 32.. of T
  float* const tXl = tXh + 128 * KX;
  float* const tTh = tXl + 128 * KX;                   // [128][32]: neurons 0..31 of T
  float* const tTl = tTh + 128 * 32;
  unsigned long long* const bars = reinterpret_cast<unsigned long long*>(tTl + 128 * 32);
  uint32_t* const tbase = reinterpret_cast<uint32_t*>(bars + 2);
  {  // the host has split and tiled both B operands (build_nnw): a straight copy
    const float4* src = reinterpret_cast<const float4*>(nnw + (tab_floats + 31) / 32 * 32);
    float4* dst = reinterpret_cast<float4*>(tB1h);
    for (int t = threadIdx.x; t < (2 * TC_NP * KP + 2 * KN * TC_NP) / 4; t += T_) cp_async16(dst + t, src + t);
    cp_async_wait_all();
  }
  const uint32_t bar_z = tc05::smem_u32(bars), bar_f = tc05::smem_u32(bars + 1);
  if (threadIdx.x < 32) tc05::tmem_alloc<TCP_TMEM_COLS>(tc05::smem_u32(tbase));
  if (threadIdx.x == 0) {
    tc05::mbar_init(bar_z, 1);
    tc05::mbar_init(bar_f, 1);
  }
  tc05::fence_smem_to_async();
  tc05::fence_before_sync();
  __syncthreads();
  tc05::fence_after_sync();
  const uint32_t tmem = *tbase;
  const uint32_t trow = tmem + ((uint32_t)(threadIdx.x & 96) << 16);  // this warp's 32 TMEM lanes
  uint32_t ph_z = 0u, ph_f = 0u;

  // a block's tiles: 128 consecutive atoms, tile index blockIdx.x + i gridDim.x (the same count for all its threads)
  const int ntiles = (n + T_ - 1) / T_;
  const float4 dummy = disp_dummy<MS::NT>();
  int t_cur = -1, t_nxt = blockIdx.x < ntiles ? (int)blockIdx.x : -1;
  float U_cur = 0.0f;  // site energy of the current tile's atom (set when its Z was consumed)
  // the head of a tile is a chain of dependent loads (mask -> count -> first displacements): requested one pass ahead
  unsigned long long mask_nx = 0ull;
  float4 pre0 = dummy, pre1 = dummy;
  if (t_nxt >= 0) {
    const int s0 = t_nxt * T_ + threadIdx.x;
    if (s0 < n) {
      mask_nx = amask[s0];
      const int c0 = __popcll(mask_nx);
      pre0 = c0 > 0 ? adisp[s0] : dummy;
      pre1 = c0 > 1 ? adisp[(size_t)npad + s0] : dummy;
    }
  }
  unsigned long long mask_cur = 0ull;

  while (t_cur >= 0 || t_nxt >= 0) {
    const bool has_cur = t_cur >= 0, has_nxt = t_nxt >= 0;  // block-uniform
    float A[NA][24];
    float U_nxt = 0.0f;
    unsigned long long mask_n = 0ull;
    // ================= forward pass and descriptor of the next tile
    if (has_nxt) {
      const int s = t_nxt * T_ + threadIdx.x;
      const bool live = s < n;  // a thread beyond the last atom carries an empty site
      const int sl = live ? s : 0;
      mask_n = live ? mask_nx : 0ull;
      const int nc = __popcll(mask_n);
      const int ti = MS::NT > 1 ? xyzt[sl].w : 0;
      float q[D];
#pragma unroll
      for (int nq = 0; nq < NR; ++nq) q[nq] = q_radial[(size_t)nq * npad + sl];
      tcp_forward<MS>(A, nc, adisp + sl, npad, pre0, pre1, mt, s_cta, ti);
#pragma unroll
      for (int nq = 0; nq < NA; ++nq) {
        float ql[4];
        tcp_q3<MS>(A, nq, ql);
#pragma unroll
        for (int l = 0; l < 4; ++l) q[NR + l * NA + nq] = ql[l];
        if (MS::B5) q[MS::B5 ? MS::V5 + nq : 0] = ql[0] * ql[0] * (1.0f / 3.0f);
        if (MS::B4) {
          float dq4[5];
          q[MS::B4 ? NR + 4 * NA + nq : 0] = tcp_q4(A[nq], dq4);
        }
      }
      if (q_out && live) {
#pragma unroll
        for (int v = 0; v < D; ++v) q_out[(size_t)v * npad + s] = q[v];
      }
#pragma unroll
      for (int v = 0; v < D; ++v) q[v] *= s_qs[v];
      if (da.dense_list && live) {  // large angular inputs: list the atom for the fp64 pass (site_fp64.cuh)
        float mx = 0.0f, mx4 = 0.0f;
#pragma unroll
        for (int v = NR; v < NR + 4 * NA; ++v) mx = fmaxf(mx, fabsf(q[v]));
#pragma unroll
        for (int v = NR + 4 * NA; v < D; ++v) mx4 = fmaxf(mx4, fabsf(q[v]));
        if (!(mx <= mt.dense_thr) || !(mx4 <= mt.dense_thr4)) da.dense_list[atomicAdd(&da.sc->dense_count, 1)] = s;
      }
      // Fp of the current tile must be complete before X's tile (which held the neurons 32.. of its T) is rewritten
      if (has_cur) {
        tc05::mbar_wait(bar_f, ph_f);
        ph_f ^= 1u;
        tc05::fence_after_sync();
      }
      char* const xh = reinterpret_cast<char*>(tXh), * const xl = reinterpret_cast<char*>(tXl);
#pragma unroll
      for (int v4 = 0; v4 < KP / 4; ++v4) {
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
    } else if (has_cur) {
      tc05::mbar_wait(bar_f, ph_f);
      ph_f ^= 1u;
      tc05::fence_after_sync();
    }

    // ================= requests whose latency the following stages hide
    const int s_c = has_cur ? t_cur * T_ + (int)threadIdx.x : 0;
    const bool live_c = has_cur && s_c < n;
    const int sl_c = live_c ? s_c : 0;
    const int nc_c = live_c ? __popcll(mask_cur) : 0;
    const float4 first_c = nc_c > 0 ? adisp[sl_c] : dummy;
    int t_nn = has_nxt ? t_nxt + (int)gridDim.x : -1;
    if (t_nn >= ntiles) t_nn = -1;
    const int s_nn = t_nn >= 0 ? t_nn * T_ + (int)threadIdx.x : n;
    mask_nx = s_nn < n ? amask[s_nn] : 0ull;

    // ================= A(nxt) in registers <-> A(cur) parked in tensor memory, four 8-column chunks per round trip
    {
      float* const Af = &A[0][0];
      constexpr int NCH = NA * 24 / 8;
#pragma unroll
      for (int g0 = 0; g0 < NCH; g0 += 4) {
        uint32_t old[4][8];
        if (has_cur) {
#pragma unroll
          for (int g = 0; g < 4; ++g)
            if (g0 + g < NCH) tc05::tmem_ld8_nowait(trow + TCP_APARK + 8 * (g0 + g), old[g]);
          tc05::wait_ld();
        }
        if (has_nxt) {
#pragma unroll
          for (int g = 0; g < 4; ++g)
            if (g0 + g < NCH) {
              uint32_t w[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) w[e] = __float_as_uint(Af[8 * (g0 + g) + e]);
              tc05::tmem_st8(trow + TCP_APARK + 8 * (g0 + g), w);
            }
        }
        if (has_cur) {
#pragma unroll
          for (int g = 0; g < 4; ++g)
            if (g0 + g < NCH) {
#pragma unroll
              for (int e = 0; e < 8; ++e) Af[8 * (g0 + g) + e] = __uint_as_float(old[g][e]);
            }
        }
      }
      if (has_nxt) tc05::wait_st();
    }

    // ================= Z(nxt) = X W0^T on the tensor core
    if (has_nxt) {
      tc05::fence_smem_to_async();
      tc05::fence_before_sync();
      __syncthreads();
      if (threadIdx.x == 0) {
        tc05::fence_after_sync();
        constexpr uint32_t id1 = tc05::idesc_tf32(128, TC_NP);
#pragma unroll
        for (int ks = 0; ks < KP / 8; ++ks) {
          const uint32_t ao = ks * 2 * 16 * 128, bo = ks * 2 * 16 * TC_NP;
          const uint64_t ah = tc05::smem_desc(tc05::smem_u32(tXh) + ao, 16 * 128, 128);
          const uint64_t al = tc05::smem_desc(tc05::smem_u32(tXl) + ao, 16 * 128, 128);
          const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB1h) + bo, 16 * TC_NP, 128);
          const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB1l) + bo, 16 * TC_NP, 128);
          tc05::mma_tf32(tmem, al, bh, id1, ks > 0);
          tc05::mma_tf32(tmem, ah, bl, id1, true);
          tc05::mma_tf32(tmem, ah, bh, id1, true);
        }
        tc05::commit(bar_z);
      }
      __syncwarp();
    }
    {  // first two displacement vectors of the tile after next (its mask has arrived by now)
      const int c0 = __popcll(mask_nx);
      pre0 = c0 > 0 ? adisp[s_nn < n ? s_nn : 0] : dummy;
      pre1 = c0 > 1 ? adisp[(size_t)npad + (s_nn < n ? s_nn : 0)] : dummy;
    }

    // ================= back-pass of the current tile (its Fp is complete: waited for above)
    if (has_cur) {
      float Fp[D];
      {
        uint32_t f[(D + 7) / 8][8];
#pragma unroll
        for (int c = 0; c < (D + 7) / 8; ++c) tc05::tmem_ld8_nowait(trow + TC_NP + 8 * c, f[c]);
        tc05::wait_ld();
#pragma unroll
        for (int v = 0; v < D; ++v) Fp[v] = __uint_as_float(f[v / 8][v % 8]) * s_qs[v];
      }
      tc05::fence_before_sync();  // the next Fp product (behind the block barrier below) overwrites these columns
      const int ti = MS::NT > 1 ? xyzt[sl_c].w : 0;
      if (live_c) {
        u_site[s_c] = U_cur;
        tcp_write_record<MS>(Fp, xyzt[s_c], s_c, ti, mt, rec);
      }
      // E[n][lm] = dU/dA[n][lm] in place
#pragma unroll
      for (int nq = 0; nq < NA; ++nq) {
        float f5 = 0.0f;
        if (MS::B5) {
          float ql[4];
          tcp_q3<MS>(A, nq, ql);
          f5 = Fp[MS::B5 ? MS::V5 + nq : 0] * (2.0f / 3.0f) * ql[0];
        }
        float dq4[5] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
        if (MS::B4) tcp_q4(A[nq], dq4);
#pragma unroll
        for (int lm = 0; lm < 24; ++lm)
          A[nq][lm] *= 2.0f * kClm[lm] * (Fp[NR + (lm_to_l(lm) - 1) * NA + nq] + (lm < 3 ? f5 : 0.0f));
        if (MS::B4) {
#pragma unroll
          for (int m5 = 0; m5 < 5; ++m5) A[nq][3 + m5] = fmaf(Fp[MS::B4 ? NR + 4 * NA + nq : 0], dq4[m5], A[nq][3 + m5]);
        }
      }
      tcp_backward<MS>(A, live_c ? mask_cur : 0ull, nc_c, adisp + sl_c, npad, first_c, mt, s_cta, ti, pforce + sl_c);
    }

    // ================= tanh layer of the next tile: Z from tensor memory, U, T = w1 (1 - h^2) -> Fp(nxt) = T W0
    if (has_nxt) {
      tc05::mbar_wait(bar_z, ph_z);
      ph_z ^= 1u;
      tc05::fence_after_sync();
      U_nxt = -mt.b1;
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        // neurons 32 half ..: half 0 -> T's own tile; half 1 -> X's tile, which the Z product has finished reading
        char* const th = reinterpret_cast<char*>(half ? tXh : tTh), * const tl = reinterpret_cast<char*>(half ? tXl : tTl);
        if (32 * half < nrow) {
          uint32_t z[32];
          tc05::tmem_ld32_nowait(trow + 32 * half, z);
          tc05::wait_ld();
#pragma unroll
          for (int m8 = 0; m8 < 32; m8 += 8) {
            if (32 * half + m8 < nrow) {  // nrow is a multiple of 8
              float4 h4[2], l4[2];
              float* hp = &h4[0].x;
              float* lp = &l4[0].x;
#pragma unroll
              for (int e = 0; e < 8; ++e) {
                const float hh = tanh_fast(__uint_as_float(z[m8 + e]));
                const float w1 = s_w1[32 * half + m8 + e];  // zero in the padding rows
                U_nxt = fmaf(w1, hh, U_nxt);
                tc05::split_tf32(w1 * fmaf(-hh, hh, 1.0f), hp[e], lp[e]);
              }
              *reinterpret_cast<float4*>(th + tc05::tile_off(128, threadIdx.x, m8)) = h4[0];
              *reinterpret_cast<float4*>(th + tc05::tile_off(128, threadIdx.x, m8 + 4)) = h4[1];
              *reinterpret_cast<float4*>(tl + tc05::tile_off(128, threadIdx.x, m8)) = l4[0];
              *reinterpret_cast<float4*>(tl + tc05::tile_off(128, threadIdx.x, m8 + 4)) = l4[1];
            }
          }
        }
      }
      tc05::fence_smem_to_async();
      tc05::fence_before_sync();
      __syncthreads();
      if (threadIdx.x == 0) {
        tc05::fence_after_sync();
        constexpr uint32_t id2 = tc05::idesc_tf32(128, KN);
        const int nks = nrow / 8;  // K steps of 8 neurons: 0..3 from T's tile, 4.. from X's
#pragma unroll 1
        for (int ks = 0; ks < nks; ++ks) {
          const bool hi_half = ks >= 4;
          const uint32_t ao = (ks & 3) * 2 * 16 * 128, bo = 2 * ks * 16 * KN;
          const uint64_t ah = tc05::smem_desc(tc05::smem_u32(hi_half ? tXh : tTh) + ao, 16 * 128, 128);
          const uint64_t al = tc05::smem_desc(tc05::smem_u32(hi_half ? tXl : tTl) + ao, 16 * 128, 128);
          const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB2h) + bo, 16 * KN, 128);
          const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB2l) + bo, 16 * KN, 128);
          tc05::mma_tf32(tmem + TC_NP, al, bh, id2, ks > 0);
          tc05::mma_tf32(tmem + TC_NP, ah, bl, id2, true);
          tc05::mma_tf32(tmem + TC_NP, ah, bh, id2, true);
        }
        tc05::commit(bar_f);
      }
      __syncwarp();
    }
    t_cur = t_nxt;
    mask_cur = mask_n;
    U_cur = U_nxt;
    t_nxt = t_nn;
  }
  tc05::fence_before_sync();
  __syncthreads();
  if (threadIdx.x < 32) tc05::tmem_dealloc<TCP_TMEM_COLS>(tmem);
}
