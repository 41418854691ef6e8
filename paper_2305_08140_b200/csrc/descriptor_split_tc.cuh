// descriptor_split_tc.cuh -- the four-lanes-per-atom kernel of LARGE models (descriptor_split.cuh; SURVEY 8(f)
// NEXT-2: the paper's own sizes) with its network layer on the tensor cores.
//
// The FFMA network is a third of k_angular_nn_split's instructions (25 rounds x (128 FMA + 16 LDS.128) per lane).  The
// tensor-core form needs rows = atoms, while the passes need four lanes per atom, so the kernel uses TWO maps of
// its 512 threads onto a tile of 128 atoms:
//   pass map     thread t <-> (atom t / 4, lane-in-quad t % 4)     forward pass, descriptor slice, records, back-pass:
//                exactly the code of k_angular_nn_split (quad shuffles, lane p owns channels p, p+4, p+8)
//   network map  warp w <-> (row quarter w % 4, neuron chunk w / 4), lane <-> row 32 (w % 4) + lane:
//                the thread reads ITS row of Z (tensor-memory lane = row, columns = its 28 neurons), takes the tanh,
//                stores its part of T, later reads its 16 columns of Fp
// and shared memory carries the data between the maps: the quads store their 16-entry descriptor slices into the
// atom's row of X (K = 64 = 4 slices), the network threads store dU/dq back as s_fp[atom][64], from which every
// quad lane reads its own slice.  Products (tc05.cuh; 3xTF32 as in k_angular_tc):
//   Z[128 x 112] = X[128 x 64] B1^T      (B1[m][16 p + idx] = w0[m][nu(p, idx)]: the slice order of SplitLayout)
//   Fp[128 x 64] = T[128 x 104] B2^T     (B2 = B1 transposed)
// One 512-thread block per SM (219 KB of shared memory: B1 / B2 hi+lo 110 KB, one 106-KB buffer that holds X, then T,
// then s_fp); the tile is long (14 neighbours x 11 channels per atom), so the three block barriers and two product
// waits per tile are a few per cent.  A[3][24] stays in registers across the network (no stash: the network needs
// no registers to speak of).  Tensor memory: Z columns [0, 112), Fp columns [128, 192) of 256.
// Shapes: four-lane models without 4-/5-body term whose slices are 16 entries (n_max 15 / 10), n_neurons <= 104.
#pragma once
#include "descriptor_split.cuh"
#include "descriptor_tc.cuh"

#define STC_THREADS 512
#define STC_NP 112   // neurons padded to the N of the first product (multiple of 16)
#define STC_KT 104   // neurons padded to the K of the second product (multiple of 8); n_neurons <= 104
#define STC_KX 64    // four slices of 16 descriptor entries
#define STC_TMEM_COLS 256
#define STC_FP_COL 128

template <class MS>
struct StcLayout {
  using LY = SplitLayout<MS>;
  static_assert(LY::SLP == 16, "four slices of 16 entries");
  // small tables (floats): b0 [nrow] | w1 [nrow] | q_scaler [4][SLS] | ctA | ctR  (the tail of SplitLayout's table)
  __host__ __device__ static constexpr int small_floats(int nrow) { return LY::table_floats(nrow) - nrow * 4 * LY::SLS; }
  // operand tiles: B1 hi/lo [112][64], B2 hi/lo [64][104], then the X / T / s_fp buffer
  static constexpr size_t b1_bytes = 2 * (size_t)STC_NP * STC_KX * 4, b2_bytes = 2 * (size_t)STC_KX * STC_KT * 4;
  static constexpr size_t xt_bytes = 2 * (size_t)128 * STC_KT * 4;
  __host__ __device__ static constexpr size_t smem_bytes(int nrow) {
    return ((size_t)small_floats(nrow) * 4 + 127) / 128 * 128 + 128 + b1_bytes + b2_bytes + xt_bytes + 4 * 128 * 4 + 64 +
           (size_t)LY::NPR * LY::NAP * 12 * 4;
  }
};

template <class MS, int AW = 1>
__global__ void __launch_bounds__(STC_THREADS, 1)
k_angular_split_tc(int n, int npad, const int4* __restrict__ xyzt,
                   const unsigned long long* __restrict__ amask, const float4* __restrict__ adisp,
                   const __grid_constant__ ModelTables<MS> mt, const float* __restrict__ nnw,
                   const float* __restrict__ q_radial, float* __restrict__ u_site,
                   AtomRec* __restrict__ rec, float4* __restrict__ pforce, float* __restrict__ q_out,
                   const DenseArgs da) {
  using LY = SplitLayout<MS>;
  using SL = StcLayout<MS>;
  static_assert(!MS::B4 && !MS::B5, "slices of 16 entries: no 4-/5-body term");
  constexpr int NT = MS::NT;
  constexpr int KA = MS::KA, NR = MS::NR, KR = MS::KR;
  constexpr int NSUB = LY::NSUB, RSUB = LY::RSUB, SLP = LY::SLP, SLS = LY::SLS, NAP = LY::NAP;
  extern __shared__ __align__(16) float smem[];
  const int nrow = LY::rows(mt.n_neurons);
  float* s_b0 = smem;                        // [nrow]
  float* s_w1 = s_b0 + nrow;                 // [nrow]
  float* s_qs = s_w1 + nrow;                 // [4][SLS]
  float* s_ct = s_qs + 4 * SLS;              // [NT*NT][NAP][KA]
  float* s_ctr = s_ct + LY::NPR * NAP * KA;  // [NT*NT][4 RSUB][KR]
  const int small = SL::small_floats(nrow);
  const uintptr_t base = (reinterpret_cast<uintptr_t>(smem + small) + 127) & ~uintptr_t(127);
  float* const tB1h = reinterpret_cast<float*>(base);
  float* const tB1l = tB1h + STC_NP * STC_KX;
  float* const tB2h = tB1l + STC_NP * STC_KX;
  float* const tB2l = tB2h + STC_KX * STC_KT;
  float* const tXT = tB2l + STC_KX * STC_KT;             // X hi [128][64] | X lo;  T hi [128][104] | T lo;  s_fp in its upper half
  float* const tXh = tXT;
  float* const tXl = tXT + 128 * STC_KX;
  float* const tTh = tXT;
  float* const tTl = tXT + 128 * STC_KT;
  float* const s_fp = tXT + 2 * 128 * STC_KX;            // [128][68] dU/dq rows, BEHIND X's region (X of the next tile may
                                                         // be stored while a slow warp still reads s_fp) inside T's
  float* const s_u = tXT + 2 * 128 * STC_KT;             // [4][128] site-energy parts per neuron chunk
  unsigned long long* const bars = reinterpret_cast<unsigned long long*>(s_u + 4 * 128);
  uint32_t* const tbase = reinterpret_cast<uint32_t*>(bars + 1);
  // the folded angular coefficients again with rows padded to 12 floats: a channel's 9 coefficients are three aligned
  // LDS.128 per neighbour instead of 27 registers held across the loops (128 registers per thread: ptxas otherwise
  // spills and sinks the next displacement load to the end of the iteration)
  float* const s_ctp = reinterpret_cast<float*>(bars + 8);  // [NT*NT][NAP][12]
  static_assert(KA <= 12, "padded coefficient rows hold 12 values");
  {
    // the small tables are the tail of SplitLayout's table (behind its w0 block); the B tiles follow the whole table
    const float4* src = reinterpret_cast<const float4*>(nnw + (size_t)nrow * 4 * SLS);
    for (int t = threadIdx.x; t < small / 4; t += STC_THREADS) cp_async16(reinterpret_cast<float4*>(smem) + t, src + t);
    const float4* bsrc = reinterpret_cast<const float4*>(nnw + (size_t)(LY::table_floats(nrow) + 31) / 32 * 32);
    float4* bdst = reinterpret_cast<float4*>(tB1h);
    for (int t = threadIdx.x; t < (int)((SL::b1_bytes + SL::b2_bytes) / 16); t += STC_THREADS) cp_async16(bdst + t, bsrc + t);
    cp_async_wait_all();
  }
  __syncthreads();
  for (int e = threadIdx.x; e < LY::NPR * NAP * 12; e += STC_THREADS) {
    const int rowc = e / 12, k = e % 12;
    s_ctp[e] = k < KA ? s_ct[rowc * KA + k] : 0.0f;
  }
  const uint32_t bar = tc05::smem_u32(bars);
  if (threadIdx.x < 32) tc05::tmem_alloc<STC_TMEM_COLS>(tc05::smem_u32(tbase));
  if (threadIdx.x == 0) tc05::mbar_init(bar, 1);
  tc05::fence_smem_to_async();
  tc05::fence_before_sync();
  __syncthreads();
  tc05::fence_after_sync();
  const uint32_t tmem = *tbase;
  uint32_t phase = 0u;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // pass map
  const int sub = lane & 3, qbase = lane & ~3;
  const unsigned qmask = 0xFu << qbase;
  const int a_loc = threadIdx.x >> 2;                    // atom of the tile this thread works on in the passes
  // network map
  const int nrow_q = warp & 3, chunk = warp >> 2;         // TMEM lane quarter of this warp, neuron chunk
  const int row = 32 * nrow_q + lane;
  const uint32_t trow = tmem + ((uint32_t)(32 * nrow_q) << 16);
  const int m_lo = 28 * chunk;                           // neurons m_lo .. m_lo + 27 (112 = 4 x 28)
  const float4 dummy = disp_dummy<NT>();
  const int ntiles = (n + 127) / 128;

  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    // ================= pass map: forward pass and descriptor slice of (atom, lane-in-quad)
    const int s = tile * 128 + a_loc;
    const bool valid = s < n;            // all 4 lanes of a quad agree; shuffles below stay inside the quad
    const int sc_ = valid ? s : 0;
    const unsigned long long mask = valid ? amask[sc_] : 0ull;
    const unsigned long long mask_hi = (AW > 1 && valid) ? amask[(size_t)npad + sc_] : 0ull;
    const int nc = __popcll(mask) + __popcll(mask_hi);
    const float4* dp = adisp + sc_;
    const int ti = NT > 1 ? xyzt[sc_].w : 0;
    float A[NSUB][24];
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] = 0.0f;
    {
      float4 nx = nc > 0 ? dp[0] : dummy;
      for (int c = 0; c < nc; ++c) {
        const float4 d = nx;
        nx = c + 1 < nc ? dp[(size_t)(c + 1) * npad] : dummy;  // in flight during this iteration
        float ux, uy, uz, r, rinv;
        unpack_disp<NT, false>(d, ux, uy, uz, r, rinv);
        float fc, T[KA], b[24];
        cheb_T_fwd<KA>(r, mt.inv_rcA, fc, T);
        eval_blm(ux, uy, uz, b);
        const float* cts = s_ctp + (NT > 1 ? (ti * NT + __float_as_int(d.w)) * NAP * 12 : 0);  // adisp.w = neighbour type
#pragma unroll
        for (int j = 0; j < NSUB; ++j) {
          float cr[12];
#pragma unroll
          for (int v4 = 0; v4 < 3; ++v4)
            *reinterpret_cast<float4*>(cr + 4 * v4) = *reinterpret_cast<const float4*>(cts + (sub + SPLIT_LANES * j) * 12 + 4 * v4);
          float g = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k) g = fmaf(cr[k], T[k], g);
          g *= fc;
#pragma unroll
          for (int lm = 0; lm < 24; ++lm) A[j][lm] = fmaf(g, b[lm], A[j][lm]);
        }
      }
    }
    {
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
#pragma unroll
      for (int i = 0; i < SLP; ++i) q[i] *= s_qs[sub * SLS + i];
      if (da.dense_list) {  // large angular inputs anywhere in the quad: list the atom for the fp64 pass (site_fp64.cuh)
        float mx = 0.0f;
#pragma unroll
        for (int i = 0; i < 4 * NSUB; ++i) mx = fmaxf(mx, fabsf(q[i]));
        const bool big = !(mx <= mt.dense_thr);
        const unsigned bq = (__ballot_sync(0xffffffffu, big) >> qbase) & 0xFu;
        if (bq && valid && sub == 0) da.dense_list[atomicAdd(&da.sc->dense_count, 1)] = s;
      }
      // this lane's slice of the atom's row of X (hi / lo), K index 16 sub + i
      char* const xh = reinterpret_cast<char*>(tXh), * const xl = reinterpret_cast<char*>(tXl);
#pragma unroll
      for (int v4 = 0; v4 < SLP / 4; ++v4) {
        float4 h4, l4;
        float* hp = &h4.x;
        float* lp = &l4.x;
#pragma unroll
        for (int e = 0; e < 4; ++e) tc05::split_tf32(valid ? q[4 * v4 + e] : 0.0f, hp[e], lp[e]);
        *reinterpret_cast<float4*>(xh + tc05::tile_off(128, a_loc, SLP * sub + 4 * v4)) = h4;
        *reinterpret_cast<float4*>(xl + tc05::tile_off(128, a_loc, SLP * sub + 4 * v4)) = l4;
      }
    }
    // ================= Z = X B1^T
    tc05::fence_smem_to_async();
    tc05::fence_before_sync();
    __syncthreads();
    if (threadIdx.x == 0) {
      tc05::fence_after_sync();
      constexpr uint32_t id1 = tc05::idesc_tf32(128, STC_NP);
#pragma unroll 1
      for (int ks = 0; ks < STC_KX / 8; ++ks) {
        const uint32_t ao = ks * 2 * 16 * 128, bo = ks * 2 * 16 * STC_NP;
        const uint64_t ah = tc05::smem_desc(tc05::smem_u32(tXh) + ao, 16 * 128, 128);
        const uint64_t al = tc05::smem_desc(tc05::smem_u32(tXl) + ao, 16 * 128, 128);
        const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB1h) + bo, 16 * STC_NP, 128);
        const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB1l) + bo, 16 * STC_NP, 128);
        tc05::mma_tf32(tmem, al, bh, id1, ks > 0);
        tc05::mma_tf32(tmem, ah, bl, id1, true);
        tc05::mma_tf32(tmem, ah, bh, id1, true);
      }
      tc05::commit(bar);
    }
    __syncwarp();
    tc05::mbar_wait(bar, phase);
    phase ^= 1u;
    tc05::fence_after_sync();

    // ================= network map: tanh layer of (row, neuron chunk); T = w1 (1 - h^2) into X's buffer (X is dead)
    {
      uint32_t z[32];
      tc05::tmem_ld32_nowait(trow + m_lo, z);  // 28 neurons of this chunk (+4 columns of the next chunk, unused)
      tc05::wait_ld();
      tc05::fence_before_sync();               // (the next tile's Z product, behind block barriers, overwrites these columns)
      char* const th = reinterpret_cast<char*>(tTh), * const tl = reinterpret_cast<char*>(tTl);
      float up = 0.0f;
#pragma unroll
      for (int m4 = 0; m4 < 28; m4 += 4) {
        float4 h4, l4;
        float* hp = &h4.x;
        float* lp = &l4.x;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int m = m_lo + m4 + e;
          float t = 0.0f;
          if (m < nrow) {                      // nrow is a multiple of 4: uniform over e
            const float hh = tanh_fast(__uint_as_float(z[m4 + e]) - s_b0[m]);
            const float w1 = s_w1[m];          // zero in the padding rows
            up = fmaf(w1, hh, up);
            t = w1 * fmaf(-hh, hh, 1.0f);
          }
          tc05::split_tf32(t, hp[e], lp[e]);
        }
        if (m_lo + m4 < STC_KT) {              // K of the second product: 104 columns
          *reinterpret_cast<float4*>(th + tc05::tile_off(128, row, m_lo + m4)) = h4;
          *reinterpret_cast<float4*>(tl + tc05::tile_off(128, row, m_lo + m4)) = l4;
        }
      }
      s_u[chunk * 128 + row] = up;
    }
    // ================= Fp = T B2^T
    tc05::fence_smem_to_async();
    tc05::fence_before_sync();
    __syncthreads();
    if (threadIdx.x == 0) {
      tc05::fence_after_sync();
      constexpr uint32_t id2 = tc05::idesc_tf32(128, STC_KX);
      const int nks = (nrow + 7) / 8;          // <= 13
#pragma unroll 1
      for (int ks = 0; ks < nks; ++ks) {
        const uint32_t ao = ks * 2 * 16 * 128, bo = ks * 2 * 16 * STC_KX;
        const uint64_t ah = tc05::smem_desc(tc05::smem_u32(tTh) + ao, 16 * 128, 128);
        const uint64_t al = tc05::smem_desc(tc05::smem_u32(tTl) + ao, 16 * 128, 128);
        const uint64_t bh = tc05::smem_desc(tc05::smem_u32(tB2h) + bo, 16 * STC_KX, 128);
        const uint64_t bl = tc05::smem_desc(tc05::smem_u32(tB2l) + bo, 16 * STC_KX, 128);
        tc05::mma_tf32(tmem + STC_FP_COL, al, bh, id2, ks > 0);
        tc05::mma_tf32(tmem + STC_FP_COL, ah, bl, id2, true);
        tc05::mma_tf32(tmem + STC_FP_COL, ah, bh, id2, true);
      }
      tc05::commit(bar);
    }
    __syncwarp();
    tc05::mbar_wait(bar, phase);
    phase ^= 1u;
    tc05::fence_after_sync();
    {  // network map: the 16 dU/dq of (row, slice = chunk) to shared memory for the quad lane that owns the slice
      float f[16];
      tc05::tmem_ld16(trow + STC_FP_COL + 16 * chunk, f);
      tc05::fence_before_sync();
#pragma unroll
      for (int v4 = 0; v4 < 4; ++v4)
        *reinterpret_cast<float4*>(s_fp + row * 68 + 16 * chunk + 4 * v4) = make_float4(f[4 * v4], f[4 * v4 + 1], f[4 * v4 + 2], f[4 * v4 + 3]);
    }
    __syncthreads();

    // ================= pass map again: dU/dq of this lane's slice, site energy, records, back-pass
    float Fp[SLP];
#pragma unroll
    for (int v4 = 0; v4 < SLP / 4; ++v4) {
      const float4 f4 = *reinterpret_cast<const float4*>(s_fp + a_loc * 68 + SLP * sub + 4 * v4);
      Fp[4 * v4 + 0] = f4.x * s_qs[sub * SLS + 4 * v4 + 0];
      Fp[4 * v4 + 1] = f4.y * s_qs[sub * SLS + 4 * v4 + 1];
      Fp[4 * v4 + 2] = f4.z * s_qs[sub * SLS + 4 * v4 + 2];
      Fp[4 * v4 + 3] = f4.w * s_qs[sub * SLS + 4 * v4 + 3];
    }
    const float U = ((s_u[a_loc] + s_u[128 + a_loc]) + (s_u[256 + a_loc] + s_u[384 + a_loc])) - mt.b1;
    {
      if (valid && sub == 0) u_site[s] = U;
      // one record per PARTNER type tp (NT > 1: d^(tp)_k = sum_n Fp_n ct^{ti tp}_nk, as k_angular_nn writes them)
#pragma unroll
      for (int tp = 0; tp < NT; ++tp) {
        float d[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) d[k] = 0.0f;
        static_assert(!MS::FPREC && KR <= 12, "large models use the 64-byte record");
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
        if (valid && sub == 0) {
          const int4 me = xyzt[s];
          float4* rp = reinterpret_cast<float4*>(rec + (size_t)NT * s + tp);
          rp[0] = make_float4(__int_as_float(me.x), __int_as_float(me.y), __int_as_float(me.z), d[0]);
          rp[1] = make_float4(d[1], d[2], d[3], d[4]);
          rp[2] = make_float4(d[5], d[6], d[7], d[8]);
          if (KR > 9 || NT > 1) rp[3] = make_float4(d[9], d[10], d[11], __int_as_float(me.w));
        }
      }
    }
    // ---- E[j][lm] = dU/dA[n_j][lm] (in place): the slice holds exactly this lane's dU/dq
#pragma unroll
    for (int j = 0; j < NSUB; ++j)
#pragma unroll
      for (int lm = 0; lm < 24; ++lm) A[j][lm] *= 2.0f * kClm[lm] * Fp[4 * j + lm_to_l(lm) - 1];

    // ---- angular partial forces dU_i/dr_ij: every lane contracts its channels, 3 numbers cross the quad
    {
      int c = 0;
      float4 nx = nc > 0 ? dp[0] : dummy;
#pragma unroll 1
      for (int mw = 0; mw < AW; ++mw)  // AW = 1 unless cap_angular > 64
      for (unsigned long long m = mw ? mask_hi : mask; m; m &= m - 1, ++c) {
        const int a = 64 * mw + __ffsll((long long)m) - 1;
        float ux, uy, uz, r, rinv;
        unpack_disp<NT, true>(nx, ux, uy, uz, r, rinv);
        const float* cts = s_ctp + (NT > 1 ? (ti * NT + __float_as_int(nx.w)) * NAP * 12 : 0);
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
          float cr[12];
#pragma unroll
          for (int v4 = 0; v4 < 3; ++v4)
            *reinterpret_cast<float4*>(cr + 4 * v4) = *reinterpret_cast<const float4*>(cts + (sub + SPLIT_LANES * j) * 12 + 4 * v4);
          float p = 0.0f, dpk = 0.0f;
#pragma unroll
          for (int k = 0; k < KA; ++k) p = fmaf(cr[k], T[k], p);
#pragma unroll
          for (int k = 1; k < KA; ++k) dpk = fmaf(cr[k], kU[k], dpk);
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
  tc05::fence_before_sync();
  __syncthreads();
  if (threadIdx.x < 32) tc05::tmem_dealloc<STC_TMEM_COLS>(tmem);
}
