// integrate.cuh -- S8: velocity-Verlet with the adaptive time step of P:77.
//   v_max = max_i |v_i(t)|;  dt = min(dt_max, max_disp / v_max)  (dt_max if v_max = 0)   [C-11]
//   v += dt/2 F/m;  x += dt v;  wrap periodic axes;  [list rebuild if needed];  F = F(x);  v += dt/2 F/m
// Master positions/velocities are fp64 in the caller's order and are integrated in place; every
// step refreshes the fixed-point compute copy (S1).  HBM-bound: ~150 B/atom per step.
// The time step and the rebuild decision stay on the device (Scalars), so a run of steps needs no
// host round trip.
#pragma once
#include "common.cuh"

// md_step arguments live on the device so that one captured CUDA graph serves every step
__global__ void k_md_params(Scalars* sc, double dt_max, double max_disp) {
  sc->dt_max = dt_max;
  sc->max_disp = max_disp;
  sc->trace_pos = 0;
}

// time step of this step from the velocity maximum left by the previous half-kick (C-11); every
// thread of k_kick_drift evaluates the same expression on the same bits
__device__ __forceinline__ double step_dt(const Scalars* sc) {
  double v2 = __longlong_as_double((long long)sc->vmax2_bits[sc->parity]);  // bits of a double >= 0
  double vmax = sqrt(v2);
  double dt = sc->dt_max;
  if (vmax > 0.0 && sc->max_disp / vmax < dt) dt = sc->max_disp / vmax;
  return dt;
}

// run by the last block of k_kick_drift: book-keeping of the step (dt for the second half-kick and the trace,
// flip the vmax slot) and the rebuild decision; in a captured graph it also sets the IF nodes
__device__ __forceinline__ void step_flag(Scalars* sc, float skin, double* dt_trace, int trace_ring,
                                          unsigned long long cond_rebuild, int use_cond) {
  double dt = step_dt(sc);
  sc->dt = dt;
  int p = sc->parity;
  sc->vmax2_bits[p ^ 1] = 0ull;
  sc->parity = p ^ 1;
  sc->n_steps += 1;
  if (dt_trace) dt_trace[sc->trace_pos % trace_ring] = dt;
  sc->trace_pos += 1;
  int r = sc->force_rebuild || top2_exceeds(sc->top2_bits, skin);
  sc->disp_sum = r ? 0.0f : top2_sum(sc->top2_bits);
  sc->top2_bits = 0ull;  // k_kick_drift of the next step accumulates the displacements since the build again
  sc->do_rebuild = r;
  sc->force_rebuild = 0;
  sc->zbl_count = 0;
  sc->dense_count = 0;
  if (r) sc->n_rebuilds += 1;
#if defined(__CUDA_ARCH__)
  if (use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)cond_rebuild, (unsigned)r);
#endif
}
struct StepFlagArgs {  // passed by value to k_kick_drift, whose last block runs step_flag
  float skin;
  double* dt_trace;
  int trace_ring;
  unsigned long long cond_rebuild;
  int use_cond;
  int n_types;
};


// ------------------------------------------------------------------ Nose-Hoover chain
// "Atoms within a thickness of 3 a0 of the boundaries ... are maintained at 300 K using the Nose-Hoover
// chain thermostat [32]".  Equations of motion of ref. [32] for the atoms of the group G
// (N_f = 3|G|, chain length M, Q_1 = N_f kT tau^2, Q_k = kT tau^2):
//   dv_i/dt = F_i/m_i - vxi_1 v_i;  dxi_k/dt = vxi_k;
//   dvxi_1/dt = (sum_G m v^2 - N_f kT)/Q_1 - vxi_1 vxi_2;  dvxi_k/dt = (Q_{k-1} vxi_{k-1}^2 - kT)/Q_k - vxi_k vxi_{k+1}.
// Splitting (C-24): NHC(dt/2) . velocity-Verlet(dt) . NHC(dt/2); NHC(delta) = descending chain
// sweep, velocity scale s = exp(-vxi_1 delta), xi += vxi delta, ascending sweep.  The chain is a handful
// of scalars: one thread advances it in fp64 after a fixed-order reduction of sum_G m v^2.
#define NEPZBL_NHC_MAX 8
struct NhcState {
  int enabled, M;
  double nf, kT, tau;
  double xi[NEPZBL_NHC_MAX], vxi[NEPZBL_NHC_MAX];
  double scale;   // s of the last NHC(delta), applied to the group's velocities by the next kernel
  double ke2;     // sum_G m v^2 (eV) the last NHC(delta) started from
  double n_group; // |G| (set by md_set_thermostat)
};

// partial[b] = sum over this block's grid-stride share of m v^2 (eV) of group atoms; cnt[b] = group atoms
__global__ void __launch_bounds__(256)
k_group_ke2_partial(int n, const double* __restrict__ vel, const int32_t* __restrict__ types,
                    const double* __restrict__ mass, const unsigned char* __restrict__ group,
                    double* __restrict__ partial, double* __restrict__ cnt) {
  __shared__ double sp[256], sn[256];
  double s = 0.0, c = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    if (group[i]) {
      double vx = vel[i], vy = vel[(size_t)n + i], vz = vel[2 * (size_t)n + i];
      s += mass[types ? types[i] : 0] * NEPZBL_AMU_A2_FS2_TO_EV * (vx * vx + vy * vy + vz * vz);
      c += 1.0;
    }
  }
  sp[threadIdx.x] = s;
  sn[threadIdx.x] = c;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sp[threadIdx.x] += sp[threadIdx.x + o];
      sn[threadIdx.x] += sn[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    partial[blockIdx.x] = sp[0];
    if (cnt) cnt[blockIdx.x] = sn[0];
  }
}

// one block: fixed-order sum of the partials, then thread 0 advances the chain by delta = dt/2.
// phase 0 (before the first half-kick): dt of THIS step = step_dt(sc) (the step's book-keeping has not run yet);
// phase 1 (after the second half-kick): dt = sc->dt.  count != NULL: only set n_group / nf (setup).
__global__ void __launch_bounds__(256)
k_nhc(const Scalars* sc, NhcState* nh, int nblocks, const double* __restrict__ partial,
      const double* __restrict__ cnt, int phase) {
  __shared__ double sp[256];
  double s = 0.0;
  const double* src = cnt ? cnt : partial;
  for (int b = threadIdx.x; b < nblocks; b += 256) s += src[b];
  sp[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sp[threadIdx.x] += sp[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x != 0) return;
  if (cnt) {
    nh->n_group = sp[0];
    nh->nf = 3.0 * sp[0];
    return;
  }
  double ke2 = sp[0];
  nh->ke2 = ke2;
  nh->scale = 1.0;
  if (!(nh->nf > 0.0)) return;
  // One NHC(delta) operator, delta = dt / 2 (equations of motion of the paper's ref. [32], reading C-24), in the
  // chain's natural units: with the inertias Q_1 = N_f kT tau^2, Q_k = kT tau^2 the driving terms reduce to
  //   link 0: (sum m v^2 / (N_f kT) - 1) / tau^2,   link 1: N_f rate_0^2 - 1 / tau^2,   link k >= 2: rate_{k-1}^2 - 1 / tau^2,
  // so no inertia is ever formed.  A link relaxes for delta / 2 under the friction of its outer neighbour (half the
  // friction, the drive, half the friction); the operator is: relax from the far end inwards, shrink the particle
  // velocities for delta, advance the thermostat positions, relax outwards again with the shrunk kinetic energy.
  const double delta = 0.5 * (phase == 0 ? step_dt(sc) : sc->dt);
  const double half = 0.5 * delta, quarter = 0.25 * delta;
  const int M = nh->M;
  const double dof = nh->nf, kT = nh->kT, inv_tau2 = 1.0 / (nh->tau * nh->tau);
  double* rate = nh->vxi;  // d xi_k / dt
  auto relax = [&](int k, double twice_ke) {
    double drive;
    if (k == 0) drive = (twice_ke / (dof * kT) - 1.0) * inv_tau2;
    else drive = (k == 1 ? dof : 1.0) * rate[k - 1] * rate[k - 1] - inv_tau2;
    const double damp = k + 1 < M ? exp(-quarter * rate[k + 1]) : 1.0;
    rate[k] = damp * (damp * rate[k] + half * drive);
  };
  for (int k = M; k-- > 0;) relax(k, ke2);
  const double sv = exp(-delta * rate[0]);
  ke2 *= sv * sv;
  for (int k = 0; k < M; ++k) nh->xi[k] += delta * rate[k];
  for (int k = 0; k < M; ++k) relax(k, ke2);
  nh->scale = sv;
}

// second NHC half-step: scale the group's velocities, then max |v|^2 over ALL atoms for the next dt
__global__ void __launch_bounds__(256)
k_scale_vmax(Scalars* sc, const NhcState* __restrict__ nh, int n, double* __restrict__ vel,
             const unsigned char* __restrict__ group) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  double v2 = 0.0;
  if (i < n) {
    const bool g = group[i] != 0;
    const double s = nh->scale;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      size_t k = (size_t)a * n + i;
      double v = vel[k];
      if (g) {
        v *= s;
        vel[k] = v;
      }
      v2 += v * v;
    }
  }
  unsigned long long b = (unsigned long long)__double_as_longlong(v2);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o);
    b = t > b ? t : b;
  }
  if ((threadIdx.x & 31) == 0 && b) atomicMax(&sc->vmax2_bits[sc->parity], b);
}

// first half-kick + drift + wrap + S1 (fixed-point copy into the sorted slot) + displacement since build
// HBM-bound (152 B per atom): all eleven loads of a thread are issued up front and six blocks share an SM at 40
// registers -- 0.337 ms (loads in program order, five blocks) -> 0.297 ms at 8.192 M atoms; eight blocks (32 registers,
// spills) 0.311 ms.
__global__ void __launch_bounds__(256, 6)
k_kick_drift(Scalars* sc, const BoxMap* __restrict__ bm, int n, double* __restrict__ pos,
             double* __restrict__ vel, const float* __restrict__ force,
             const int32_t* __restrict__ types, const double* __restrict__ inv_mass,
             const int* __restrict__ inv_perm, int4* __restrict__ xyzt,
             const int4* __restrict__ xyzt_build, const unsigned char* __restrict__ group,
             const NhcState* __restrict__ nh, const StepFlagArgs fa) {
  __shared__ unsigned sh[64];
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.0f;
  if (i < n) {
    const double dt = step_dt(sc);
    const double sg = (group && group[i]) ? nh->scale : 1.0;  // first NHC(dt/2) of the step (k_nhc)
    int t = checked_type(sc, types, i, fa.n_types);
    double im = inv_mass[t];  // 1 / (m * 103.6426965): acceleration in A/fs^2 per eV/A
    unsigned int u[3];
    double xn[3];
    bool finite = true;
    // every load of the thread is issued before the first use (the kernel waits on memory latency, nothing else)
    double v_in[3], x_in[3];
    float f_in[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      size_t k = (size_t)a * n + i;
      v_in[a] = vel[k];
      x_in[a] = pos[k];
      f_in[a] = force[k];
    }
    const int s = inv_perm[i];
    const int4 b = xyzt_build[i];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      size_t k = (size_t)a * n + i;
      double v = v_in[a];
      if (group) v *= sg;
      v += 0.5 * dt * ((double)f_in[a] * im);
      double xx = x_in[a] + dt * v;
      if (!bm->tri && bm->pbc[a]) xx -= bm->L[a] * floor(xx / bm->L[a]);
      vel[k] = v;
      xn[a] = xx;
      finite = finite && isfinite(xx);
    }
    if (bm->tri && finite) {  // wrap along the lattice vectors: s = x H^-1, s -= floor(s), x = s H
      double sf[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        sf[a] = xn[0] * bm->Hi[a] + xn[1] * bm->Hi[3 + a] + xn[2] * bm->Hi[6 + a];
        sf[a] -= floor(sf[a]);
      }
#pragma unroll
      for (int b = 0; b < 3; ++b) xn[b] = sf[0] * bm->H[b] + sf[1] * bm->H[3 + b] + sf[2] * bm->H[6 + b];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) pos[(size_t)a * n + i] = xn[a];
    if (!finite) {
      sc->nonfinite = 1;
      xn[0] = xn[1] = xn[2] = 0.0;
    }
    fix_position(bm, xn[0], xn[1], xn[2], u);
    NZ_CHECK((unsigned)s < (unsigned)n, "k_kick_drift: sorted slot outside [0, n)");
    xyzt[s] = make_int4((int)u[0], (int)u[1], (int)u[2], t);
    float dx, dy, dz;
    fixed_disp_rt(bm, (int)u[0] - b.x, (int)u[1] - b.y, (int)u[2] - b.z, dx, dy, dz);
    d2 = dx * dx + dy * dy + dz * dz;
  }
  const Top2 m = block_top2(d2, sh);
  if (threadIdx.x == 0) {
    top2_publish(&sc->top2_bits, m);
    // the block that finishes last does the step's book-keeping (formerly a one-thread kernel of its own):
    // every other block has read dt / parity and published its displacement maximum before its ticket
    __threadfence();
    if (atomicAdd(&sc->blocks_done, 1u) == gridDim.x - 1) {
      __threadfence();
      sc->blocks_done = 0u;
      step_flag(sc, fa.skin, fa.dt_trace, fa.trace_ring, fa.cond_rebuild, fa.use_cond);
    }
  }
}

// second half-kick; leaves max |v|^2 for the next step's dt (integer atomicMax on the bits of a
// non-negative double is order-independent)
__global__ void __launch_bounds__(256)
k_kick(Scalars* sc, int n, double* __restrict__ vel,
       const float* __restrict__ force, const int32_t* __restrict__ types,
       const double* __restrict__ inv_mass, int do_kick, int do_vmax) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  double v2 = 0.0;
  if (i < n) {
    const double dt = sc->dt;
    double im = inv_mass[types ? types[i] : 0];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      size_t k = (size_t)a * n + i;
      double v = vel[k];
      if (do_kick) {
        v += 0.5 * dt * ((double)force[k] * im);
        vel[k] = v;
      }
      v2 += v * v;
    }
  }
  unsigned long long b = (unsigned long long)__double_as_longlong(v2);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o);
    b = t > b ? t : b;
  }
  if (do_vmax && (threadIdx.x & 31) == 0 && b) atomicMax(&sc->vmax2_bits[sc->parity], b);
}

// fixed-order fp64 reductions for md_energies: per-block tree -> partial[block]; then one block.
__global__ void __launch_bounds__(256)
k_energy_partial(int n, const double* __restrict__ vel, const double* __restrict__ energy,
                 const int32_t* __restrict__ types, const double* __restrict__ mass,
                 double* __restrict__ partial) {
  __shared__ double sp[256], sk[256];
  double ep = 0.0, ek = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    double vx = vel[i], vy = vel[(size_t)n + i], vz = vel[2 * (size_t)n + i];
    ek += 0.5 * mass[types ? types[i] : 0] * NEPZBL_AMU_A2_FS2_TO_EV * (vx * vx + vy * vy + vz * vz);
    ep += energy[i];
  }
  sp[threadIdx.x] = ep;
  sk[threadIdx.x] = ek;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sp[threadIdx.x] += sp[threadIdx.x + o];
      sk[threadIdx.x] += sk[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    partial[2 * blockIdx.x] = sp[0];
    partial[2 * blockIdx.x + 1] = sk[0];
  }
}
__global__ void __launch_bounds__(256)
k_energy_final(int nblocks, const double* __restrict__ partial, double* __restrict__ out) {
  __shared__ double sp[256], sk[256];
  double ep = 0.0, ek = 0.0;
  if (nblocks < 0) {  // single array of -nblocks partial sums -> out[0]
    for (int b = threadIdx.x; b < -nblocks; b += 256) ep += partial[b];
  } else {
    for (int b = threadIdx.x; b < nblocks; b += 256) {
      ep += partial[2 * b];
      ek += partial[2 * b + 1];
    }
  }
  sp[threadIdx.x] = ep;
  sk[threadIdx.x] = ek;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sp[threadIdx.x] += sp[threadIdx.x + o];
      sk[threadIdx.x] += sk[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out[0] = sp[0];
    out[1] = sk[0];
  }
}
