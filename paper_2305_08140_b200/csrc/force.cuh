// force.cuh -- S7 (force / virial accumulation, gather form) and S5 (ZBL pair term).
//
// S7:  F_i = sum_j (dU_i/dr_ij - dU_j/dr_ji),  W_i = sum_j r_ij (x) dU_j/dr_ji.
//   radial part:  dU_i/dr_ij = rhat_ij sum_k d_i[k] (f_c T_k)'(r_ij), d_i[k] = sum_n Fp_i[n] ct_nk,
//                 so F_i += rhat_ij sum_k (d_i[k] + d_j[k]) (f_c T_k)'.  Per pair the neighbour's
//                 record {position, d_j} (AtomRec, one 128-byte line) is gathered with a 256-bit
//                 (LDG.E.256, new on sm_100) and a 128-bit load;
//   angular part: partial forces stored by k_angular_nn; F_i += p[i][a] - p[j][rev[i][a]].
//   Gather form only: every atom sums its own pairs in list order -> no float atomics, bitwise
//   reproducible.
// S5 (Eq. 1-4; switch P:71): evaluated in FP64 from the fp64 master positions, only for
//   atoms flagged by k_radial as having a neighbour inside r_outer (rare: none in a thermal lattice).
#pragma once
#include "descriptor.cuh"

// FORCE_LANES lanes per atom: lane p takes list entries p, p+4, ... of both lists (skipping ahead to the
// next radial entry inside the cutoff before the convergent body); F and W are combined over the 4
// lanes by a fixed-order shuffle tree, so the result is still bit-reproducible.
#define FORCE_LANES 4
// MD steps fuse the second half-kick of velocity-Verlet (S8b) into this kernel's epilogue (KickArgs::vel != NULL):
// v += dt/2 F/m and max |v|^2 for the next step's dt, as k_kick does.  Atoms with a neighbour inside the ZBL
// range are left to k_zbl, which adds the pair force first and then kicks them itself (their force is not final
// here); the test is k_radial's, on the same bits.  In a captured graph thread 0 also opens / closes the IF
// node of k_zbl (zbl_count is final once k_radial has run).
struct KickArgs {
  Scalars* sc;
  double* vel;               // NULL: no kick (plain evaluation)
  const double* inv_mass;
  int do_vmax;               // 0 when a thermostat rescales the velocities afterwards (k_scale_vmax)
  unsigned long long cond_zbl;
  int use_cond;
};
// BLK = threads per block (32 or 64, chosen by the host from the grid size; a template parameter because the code
// ptxas generates under __launch_bounds__(32) is 2 % faster than the same source under a bound of 64 or 128)
template <class MS, bool VIRIAL, int BLK, bool TRI, int AW = 1>
__global__ void __launch_bounds__(BLK, (MS::NT > 1 && MS::FPREC) ? 1024 / BLK : 0)
k_force(const BoxMap* __restrict__ bm, int n, int npad, const int4* __restrict__ xyzt,
        const int* __restrict__ nn_r, const int* __restrict__ nl_r, const int* __restrict__ nn_a,
        const int* __restrict__ nl_a, const unsigned char* __restrict__ rev,
        const __grid_constant__ ModelTables<MS> mt, const AtomRec* __restrict__ rec,
        const unsigned* __restrict__ rmask, const unsigned* __restrict__ tmask, int mask_words, const unsigned long long* __restrict__ amask, const float4* __restrict__ pforce, const float* __restrict__ u_site,
        const int* __restrict__ perm, double* __restrict__ energy, float* __restrict__ force,
        float* __restrict__ virial, const KickArgs ka) {
  constexpr int KR = MS::KR;
#if defined(__CUDA_ARCH__)
  if (ka.use_cond && blockIdx.x == 0 && threadIdx.x == 0)
    cudaGraphSetConditional((cudaGraphConditionalHandle)ka.cond_zbl, ka.sc->zbl_count > 0 ? 1u : 0u);
#endif
  bool close = false;
  static_assert(KR <= 12, "AtomRec holds 12 coefficients");
  const int gt = blockIdx.x * blockDim.x + threadIdx.x;
  const int s = gt / FORCE_LANES, sub = gt % FORCE_LANES;
  const bool valid = s < n;
  const int sc_ = valid ? s : 0;
  constexpr int NR = MS::NR;
  constexpr int NT = MS::NT;
  struct Rec { int ux, uy, uz, type; float d[12]; };  // d[] holds Fp[0..4] when MS::FPREC
  // NT > 1: the records are rec[NT * atom + partner type] (k_angular_nn): the coefficients of `atom` as the central
  // atom of a pair with a neighbour of that type; the record also carries the atom's own type
  auto load = [&](Rec& r, int idx, int partner_type) {
    r.type = 0;
    if (MS::FPREC) ld_rec32(rec, idx, r.ux, r.uy, r.uz, r.d);
    else {
      const AtomRec* p = rec + (size_t)NT * idx + (NT > 1 ? partner_type : 0);
      ld_rec(p, r.ux, r.uy, r.uz, r.d, KR);
      if (NT > 1) r.type = ld_rec_type(p);
    }
  };
  // d[k] = sum_n Fp[n] ct_nk from a 32-byte record's Fp
  auto contract = [&](const float* fp, float* d) {
#pragma unroll
    for (int k = 0; k < KR; ++k) {
      float t = 0.0f;
#pragma unroll
      for (int nq = 0; nq < NR; ++nq) t = fmaf(fp[nq < 12 ? nq : 0], mt.ctR[0][nq][k], t);
      d[k] = t;
    }
  };
  // NT > 1 with 32-byte records {position, Fp}: the folded radial coefficients of all ordered type pairs in shared
  // memory, rows padded to 12 floats (three aligned LDS.128 per row: the table of (neighbour type, my type) is picked per pair)
  __shared__ __align__(16) float s_ctr[(NT > 1 && MS::FPREC) ? NT * NT * NR * 12 : 4];
  if (NT > 1 && MS::FPREC) {
    for (int e = threadIdx.x; e < NT * NT * NR * 12; e += BLK) {
      const int pr = e / (NR * 12), nq = (e / 12) % NR, k = e % 12;
      s_ctr[e] = k < KR ? mt.ctR[pr][nq][k] : 0.0f;
    }
    __syncthreads();
  }
  // d[k] = sum_n fp[n] ct^{pair}_nk from that table
  auto contract_pair = [&](const float* fp, int pair, float* d) {
#pragma unroll
    for (int k = 0; k < KR; ++k) d[k] = 0.0f;
#pragma unroll
    for (int nq = 0; nq < NR; ++nq) {
      float c[12];
#pragma unroll
      for (int v4 = 0; v4 < 3; ++v4)
        *reinterpret_cast<float4*>(c + 4 * v4) = *reinterpret_cast<const float4*>(s_ctr + (pair * NR + nq) * 12 + 4 * v4);
#pragma unroll
      for (int k = 0; k < KR; ++k) d[k] = fmaf(fp[nq], c[k], d[k]);
    }
  };
  Rec me;
  load(me, sc_, 0);
  const int ti = (NT > 1 && MS::FPREC) ? xyzt[sc_].w : me.type;
  float me_d1[NT > 1 ? 12 : 1];  // my coefficients towards a neighbour of type 1 (me.d / me_d0: towards type 0)
  float me_d0[(NT > 1 && MS::FPREC) ? 12 : 1];
  if (NT > 1) {
    static_assert(NT <= 2, "k_force keeps one coefficient set per partner type in registers");
    if (MS::FPREC) {  // d_i^(t)[k] = sum_n Fp_i[n] ct^{ti t}_nk for both partner types, once per atom
      contract_pair(me.d, ti * NT + 0, me_d0);
      contract_pair(me.d, ti * NT + 1, me_d1);
    } else {
      Rec t1;
      load(t1, sc_, 1);
#pragma unroll
      for (int k = 0; k < 12; ++k) me_d1[NT > 1 ? k : 0] = t1.d[k];
    }
  }
  float hm[9];  // fixed-point difference -> Cartesian displacement (only the diagonal is live for orthogonal boxes)
#pragma unroll
  for (int k = 0; k < 9; ++k) hm[k] = (TRI || k % 4 == 0) ? bm->hm[k] : 0.0f;
  float fx = 0.0f, fy = 0.0f, fz = 0.0f;
  float w[9];
#pragma unroll
  for (int c = 0; c < 9; ++c) w[c] = 0.0f;

  // ---- radial pairs: only the entries k_radial found inside the cutoff (bit mask per lane), with the
  //      next entry's index and record gathers in flight while the current pair is evaluated
  {
    const int* lp = nl_r + nl_at(sub, sc_, npad);  // rows sub, sub + 4, ...: lstride apart
    const size_t lstride = (size_t)FORCE_LANES * npad;
    int word = 0;
    constexpr bool TM = NT > 1 && MS::FPREC;  // neighbour types from k_radial's type mask (the 32-byte record has none)
    unsigned m = valid ? rmask[(size_t)sub * npad + sc_] : 0u;
    unsigned tm = (TM && valid) ? tmask[(size_t)sub * npad + sc_] : 0u;
    int t_pop = 0;  // type of the entry next_j() returned last
    // pop the next entry of this lane: returns its neighbour index or -1
    auto next_j = [&]() -> int {
      while (m == 0u) {
        if (++word >= mask_words) return -1;
        m = valid ? rmask[((size_t)word * FORCE_LANES + sub) * npad + sc_] : 0u;
        if (TM) tm = valid ? tmask[((size_t)word * FORCE_LANES + sub) * npad + sc_] : 0u;
      }
      int b = __ffs((int)m) - 1;
      m &= m - 1u;
      if (TM) t_pop = (tm >> b) & 1u;
      const int* a = lp + (size_t)(32 * word + b) * lstride;
      // Small systems (BLK == 32: the lists live in the L2): the lane's entry after next -- the in-cutoff entries are a
      // dense prefix, so almost always two rows on -- is prefetched into the L1: k_force 78.6 -> 73.7 us at 128 000
      // atoms.  At 8.192 M atoms, where the lists stream from DRAM, the same prefetch (L1 or L2) costs 3 %, and
      // loading the entries two pairs ahead instead of one 2.5 %: not done there.
      if (BLK == 32) prefetch_l1(a + 2 * lstride);
      return *a;
    };
    int j_cur = next_j();
    int t_cur = t_pop;
    Rec o_cur, o_nxt;
    load(o_cur, j_cur >= 0 ? j_cur : sc_, ti);
    int j_nxt = j_cur >= 0 ? next_j() : -1;
    int t_nxt = t_pop;
    while (j_cur >= 0) {
      NZ_CHECK(j_cur < n && j_nxt < n, "k_force: radial list entry outside [0, n)");
      load(o_nxt, j_nxt >= 0 ? j_nxt : sc_, ti);
      int j_nn = j_nxt >= 0 ? next_j() : -1;
      const int t_nn = t_pop;
      const Rec& o = o_cur;
      const int tj = TM ? t_cur : o.type;
      float dx, dy, dz;
      fixed_disp<TRI>(hm, o.ux - me.ux, o.uy - me.uy, o.uz - me.uz, dx, dy, dz);
      float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
      close = close || (r2 < mt.zbl_flag_r2);
      float rinv = rsqrt_fast(r2), r = r2 * rinv;
      float fc, dfc, x, dxdr, T[KR], Uc[KR];
      cheb_T<KR>(r, mt.inv_rcR, fc, dfc, x, dxdr, T);
      cheb_U<KR>(x, Uc);
      // sum_k d[k] (f_c T_k)' = f_c' sum_k d[k] T_k + f_c x' sum_{k>=1} d[k] k U_{k-1}
      const float e = fc * dxdr;
      float gi, gj = 0.0f;
      if (VIRIAL) {
        float ai = 0.0f, bi = 0.0f, aj = 0.0f, bj = 0.0f;
        float di[KR], dj[KR];
        if (TM) {
          contract_pair(o.d, tj * NT + ti, dj);
#pragma unroll
          for (int k = 0; k < KR; ++k) di[k] = tj == 1 ? me_d1[NT > 1 ? k : 0] : me_d0[TM ? k : 0];
        } else if (MS::FPREC) {
          contract(me.d, di);
          contract(o.d, dj);
        } else {
#pragma unroll
          for (int k = 0; k < KR; ++k) {
            di[k] = (NT > 1 && tj == 1) ? me_d1[NT > 1 ? k : 0] : me.d[k];
            dj[k] = o.d[k];
          }
        }
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
        gi = fmaf(dfc, ai, e * bi);  // dU_i/dr along rhat_ij
        gj = fmaf(dfc, aj, e * bj);  // dU_j/dr along rhat_ji (same scalar form)
      } else {
        // forces only need g_i + g_j: contract once with d_i + d_j (two partial sums each for ILP)
        float a0 = 0.0f, a1 = 0.0f, b0 = 0.0f, b1 = 0.0f;
        float dsum[KR];
        if (TM) {
          contract_pair(o.d, tj * NT + ti, dsum);
#pragma unroll
          for (int k = 0; k < KR; ++k) dsum[k] += tj == 1 ? me_d1[NT > 1 ? k : 0] : me_d0[TM ? k : 0];
        } else if (MS::FPREC) {
          float fs5[5];
#pragma unroll
          for (int nq = 0; nq < 5; ++nq) fs5[nq] = me.d[nq] + o.d[nq];
          contract(fs5, dsum);
        } else {
#pragma unroll
          for (int k = 0; k < KR; ++k) dsum[k] = ((NT > 1 && tj == 1) ? me_d1[NT > 1 ? k : 0] : me.d[k]) + o.d[k];
        }
#pragma unroll
        for (int k = 0; k < KR; ++k) {
          float ds = dsum[k];
          if (k & 1) a1 = fmaf(ds, T[k], a1); else a0 = fmaf(ds, T[k], a0);
          if (k >= 1) {
            float ku = (float)k * Uc[k - 1];
            if (k & 1) b1 = fmaf(ds, ku, b1); else b0 = fmaf(ds, ku, b0);
          }
        }
        gi = fmaf(dfc, a0 + a1, e * (b0 + b1));
      }
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
      j_cur = j_nxt;
      o_cur = o_nxt;
      j_nxt = j_nn;
      t_cur = t_nxt;
      t_nxt = t_nn;
    }
  }

  // ---- angular pairs inside the cutoff (bit mask from k_angular_nn; by symmetry of r_ij the reverse
  //      entry is in j's mask too): own partial force minus the neighbour's partial force on the same
  //      pair.  Lane p takes the in-cutoff entries number p, p+4, ...; 2 entries per lane per iteration
  //      so that the dependent gathers overlap.
  {
    // the in-cutoff entries in list order: word 0 of the mask, then (cap_angular > 64 only) word 1; TWO selects the
    // two-word walk -- the common one-word case keeps its plain bit arithmetic
    auto angular_part = [&](auto two) {
    constexpr bool TWO = decltype(two)::value;
    unsigned long long m = valid ? amask[sc_] : 0ull;
    unsigned long long m_hi = (TWO && valid) ? amask[(size_t)npad + sc_] : 0ull;
    int abase = 0;
    auto drop = [&]() {  // remove the lowest set bit
      m &= m - 1;
      if (TWO && m == 0ull && m_hi != 0ull) { m = m_hi; m_hi = 0ull; abase = 64; }
    };
    if (TWO && m == 0ull && m_hi != 0ull) { m = m_hi; m_hi = 0ull; abase = 64; }
    for (int k = 0; k < sub; ++k) drop();  // the entries of the lanes below
    while (m) {
      const int a0 = abase + __ffsll((long long)m) - 1;
      drop(); drop(); drop(); drop();
      const bool ok1 = m != 0ull;
      const int a1 = ok1 ? abase + __ffsll((long long)m) - 1 : a0;
      drop(); drop(); drop(); drop();
      const size_t e0 = (size_t)a0 * npad + sc_, e1 = (size_t)a1 * npad + sc_;
      int j0 = nl_a[nl_at(a0, sc_, npad)], j1 = nl_a[nl_at(a1, sc_, npad)];
      int b0 = rev[e0], b1 = rev[e1];
      NZ_CHECK((unsigned)j0 < (unsigned)n && (unsigned)j1 < (unsigned)n, "k_force: angular list entry outside [0, n)");
      NZ_CHECK((b0 == 255 || b0 < 64 * AW) && (b1 == 255 || b1 < 64 * AW), "k_force: reverse slot");
      float4 pij0 = pforce[e0], pij1 = pforce[e1];
      // rev == 255: j's list does not hold i -- only after a neighbour-capacity overflow (j's list was dropped and
      // the call reports NEPZBL_E_NEIGHBOR_OVERFLOW); the value must never be used as a row index
      const float4 zero4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      float4 pji0 = b0 != 255 ? pforce[(size_t)b0 * npad + j0] : zero4;
      float4 pji1 = b1 != 255 ? pforce[(size_t)b1 * npad + j1] : zero4;
      if (!ok1) pij1 = pji1 = zero4;
      fx += pij0.x - pji0.x;
      fy += pij0.y - pji0.y;
      fz += pij0.z - pji0.z;
      fx += pij1.x - pji1.x;
      fy += pij1.y - pji1.y;
      fz += pij1.z - pji1.z;
      if (VIRIAL) {
        int4 o0 = xyzt[j0], o1 = xyzt[j1];
        {
          float dx, dy, dz;
          fixed_disp<TRI>(hm, o0.x - me.ux, o0.y - me.uy, o0.z - me.uz, dx, dy, dz);
          w[0] = fmaf(dx, pji0.x, w[0]); w[1] = fmaf(dx, pji0.y, w[1]); w[2] = fmaf(dx, pji0.z, w[2]);
          w[3] = fmaf(dy, pji0.x, w[3]); w[4] = fmaf(dy, pji0.y, w[4]); w[5] = fmaf(dy, pji0.z, w[5]);
          w[6] = fmaf(dz, pji0.x, w[6]); w[7] = fmaf(dz, pji0.y, w[7]); w[8] = fmaf(dz, pji0.z, w[8]);
        }
        {
          float dx, dy, dz;
          fixed_disp<TRI>(hm, o1.x - me.ux, o1.y - me.uy, o1.z - me.uz, dx, dy, dz);
          w[0] = fmaf(dx, pji1.x, w[0]); w[1] = fmaf(dx, pji1.y, w[1]); w[2] = fmaf(dx, pji1.z, w[2]);
          w[3] = fmaf(dy, pji1.x, w[3]); w[4] = fmaf(dy, pji1.y, w[4]); w[5] = fmaf(dy, pji1.z, w[5]);
          w[6] = fmaf(dz, pji1.x, w[6]); w[7] = fmaf(dz, pji1.y, w[7]); w[8] = fmaf(dz, pji1.z, w[8]);
        }
      }
    }
    };
    angular_part(std::integral_constant<bool, (AW > 1)>{});
  }

  // ---- combine the 4 lanes (fixed order), results in the caller's atom order
  fx += __shfl_xor_sync(0xffffffffu, fx, 1); fx += __shfl_xor_sync(0xffffffffu, fx, 2);
  fy += __shfl_xor_sync(0xffffffffu, fy, 1); fy += __shfl_xor_sync(0xffffffffu, fy, 2);
  fz += __shfl_xor_sync(0xffffffffu, fz, 1); fz += __shfl_xor_sync(0xffffffffu, fz, 2);
  if (VIRIAL) {
#pragma unroll
    for (int c = 0; c < 9; ++c) {
      w[c] += __shfl_xor_sync(0xffffffffu, w[c], 1);
      w[c] += __shfl_xor_sync(0xffffffffu, w[c], 2);
    }
  }
  const unsigned cb = __ballot_sync(0xffffffffu, close);
  const int i = valid ? perm[s] : 0;
  if (ka.vel) {  // S8b (uniform branch): lane a < 3 of the quad kicks component a; |v|^2 = (vx^2 + vy^2) + vz^2
    const bool mine = valid && !((cb >> (threadIdx.x & 28)) & 0xFu);
    double v = 0.0;
    if (mine && sub < 3) {
      const double dt = ka.sc->dt;
      const double im = ka.inv_mass[xyzt[s].w];
      const float fa = sub == 0 ? fx : (sub == 1 ? fy : fz);
      const size_t k = (size_t)sub * n + i;
      v = ka.vel[k] + 0.5 * dt * ((double)fa * im);
      ka.vel[k] = v;
    }
    double v2 = v * v;
    const double vy2 = __shfl_down_sync(0xffffffffu, v2, 1), vz2 = __shfl_down_sync(0xffffffffu, v2, 2);
    v2 = (v2 + vy2) + vz2;  // meaningful on lane 0 of each quad
    unsigned long long b = (ka.do_vmax && mine && sub == 0) ? (unsigned long long)__double_as_longlong(v2) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o);
      b = t > b ? t : b;
    }
    if ((threadIdx.x & 31) == 0 && b) {
      unsigned long long* slot = &ka.sc->vmax2_bits[ka.sc->parity];
      if (b > *(volatile unsigned long long*)slot) atomicMax(slot, b);
    }
  }
  if (!valid) return;
  if (sub == 0 && energy) energy[i] = (double)u_site[s];
  if (force) {
    if (sub == 0) force[i] = fx;
    if (sub == 1) force[(size_t)n + i] = fy;
    if (sub == 2) force[2 * (size_t)n + i] = fz;
  }
  if (VIRIAL) {
#pragma unroll
    for (int c = 0; c < 9; ++c)
      if ((c & 3) == sub) virial[(size_t)c * n + i] = w[c];
  }
}

// minimum image of a Cartesian difference in fp64: per periodic axis for orthogonal boxes, along the lattice vectors
// (s = d H^-1, s -= rint(s), d = s H) for triclinic ones; exact for pairs closer than half the smallest cell height
__device__ __forceinline__ void min_image_f64(const BoxMap* __restrict__ bm, double d[3]) {
  if (bm->tri) {
    double sf[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      sf[a] = d[0] * bm->Hi[a] + d[1] * bm->Hi[3 + a] + d[2] * bm->Hi[6 + a];
      sf[a] -= rint(sf[a]);
    }
#pragma unroll
    for (int b = 0; b < 3; ++b) d[b] = sf[0] * bm->H[b] + sf[1] * bm->H[3 + b] + sf[2] * bm->H[6 + b];
  } else {
#pragma unroll
    for (int a = 0; a < 3; ++a)
      if (bm->pbc[a]) d[a] -= bm->L[a] * rint(d[a] / bm->L[a]);
  }
}

struct ZblParams {
  double r_inner, r_outer;
  int n_terms;
  double c[4], d[4];
  double a_num, a_pow, coulomb_k;
  double Z[8];
  double Zpow[8];   // Z^a_pow (Eq. 4), evaluated once on the host
  float filter_r2;  // fixed-point prefilter radius^2
};

// S5: U_ZBL = K Z_i Z_j / r * phi(r/a) * f_c(r)   (Eq. 2-4), half to each atom (Eq. 1).
// Adds to energy / force / virial of the flagged atoms.  ZBL_LANES lanes share an atom (neighbour k goes to lane
// k mod 8; fixed-order xor butterfly at the end, so the sums are reproducible): a thread per atom walked its ~90 list
// entries alone, one dependent gather after the other (0.08 ms for the 7 000 flagged atoms of a developed cascade).
#define ZBL_LANES 8
__global__ void __launch_bounds__(64)
k_zbl(const Scalars* sc, const BoxMap* __restrict__ bm, const int* __restrict__ zbl_list, int n,
      int npad, const int4* __restrict__ xyzt, const int* __restrict__ nn_r,
      const int* __restrict__ nl_r, const int* __restrict__ perm, const double* __restrict__ pos,
      const ZblParams zp, double* __restrict__ energy, float* __restrict__ force,
      float* __restrict__ virial, const KickArgs ka) {
  const int total = sc->zbl_count;
  const int sub = threadIdx.x % ZBL_LANES;
  const unsigned gmask = ((1u << ZBL_LANES) - 1u) << ((threadIdx.x & 31) / ZBL_LANES * ZBL_LANES);
  for (int t = (blockIdx.x * blockDim.x + threadIdx.x) / ZBL_LANES; t < total; t += gridDim.x * blockDim.x / ZBL_LANES) {
    int s = zbl_list[t];
    NZ_CHECK((unsigned)s < (unsigned)n, "k_zbl: flagged atom outside [0, n)");
    int i = perm[s];
    const int4 me = xyzt[s];
    double xi = pos[i], yi = pos[(size_t)n + i], zi = pos[2 * (size_t)n + i];
    double e = 0.0, f[3] = {0.0, 0.0, 0.0}, w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    int cnt = nn_r[s];
    for (int k = sub; k < cnt; k += ZBL_LANES) {
      int j = nl_r[nl_at(k, s, npad)];
      NZ_CHECK((unsigned)j < (unsigned)n, "k_zbl: list entry outside [0, n)");
      int4 o = xyzt[j];
      float fdx, fdy, fdz;
      fixed_disp_rt(bm, o.x - me.x, o.y - me.y, o.z - me.z, fdx, fdy, fdz);
      if (fdx * fdx + fdy * fdy + fdz * fdz >= zp.filter_r2) continue;
      int jj = perm[j];
      double d[3] = {pos[jj] - xi, pos[(size_t)n + jj] - yi, pos[2 * (size_t)n + jj] - zi};
      min_image_f64(bm, d);  // minimum image in fp64
      double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      if (!(r < zp.r_outer)) continue;
      double Zi = zp.Z[me.w], Zj = zp.Z[o.w];
      double a0 = zp.a_num / (zp.Zpow[me.w] + zp.Zpow[o.w]);  // Eq. 4
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
#pragma unroll
    for (int o = 1; o < ZBL_LANES; o <<= 1) {
      e += __shfl_xor_sync(gmask, e, o);
#pragma unroll
      for (int a = 0; a < 3; ++a) f[a] += __shfl_xor_sync(gmask, f[a], o);
      if (virial) {
#pragma unroll
        for (int c = 0; c < 9; ++c) w[c] += __shfl_xor_sync(gmask, w[c], o);
      }
    }
    if (sub != 0) continue;
    if (energy) energy[i] += e;
    double v2 = 0.0;
    if (force)
      for (int a = 0; a < 3; ++a) {
        const float ft = (float)((double)force[(size_t)a * n + i] + f[a]);
        force[(size_t)a * n + i] = ft;
        if (ka.vel) {  // S8b for the atoms k_force left out (their force is final only now)
          double v = ka.vel[(size_t)a * n + i] + 0.5 * ka.sc->dt * ((double)ft * ka.inv_mass[me.w]);
          ka.vel[(size_t)a * n + i] = v;
          v2 += v * v;
        }
      }
    if (ka.vel && ka.do_vmax && v2 > 0.0)
      atomicMax(&ka.sc->vmax2_bits[ka.sc->parity], (unsigned long long)__double_as_longlong(v2));
    if (virial)
      for (int c = 0; c < 9; ++c) virial[(size_t)c * n + i] = (float)((double)virial[(size_t)c * n + i] + w[c]);
  }
}

// descriptor export (parity tests): [D][npad] sorted -> [n][D] caller order
__global__ void k_export_q(int n, int npad, int D, const int* __restrict__ qmap, const int* __restrict__ perm,
                           const float* __restrict__ q_sorted, float* __restrict__ out) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int i = perm[s];
  // qmap: component v of the caller's model is component qmap[v] of the kernel shape (identity unless padded)
  for (int v = 0; v < D; ++v) out[(size_t)i * D + v] = q_sorted[(size_t)qmap[v] * npad + s];
}
