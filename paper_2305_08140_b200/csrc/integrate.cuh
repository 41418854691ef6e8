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

// one thread, after k_kick_drift: book-keeping of the step (dt for the second half-kick and the trace,
// flip the vmax slot) and the rebuild decision; in a captured graph it also sets the IF nodes
__global__ void k_step_flag(Scalars* sc, float half_skin2, double* dt_trace, int trace_ring,
                            unsigned long long cond_rebuild, int use_cond) {
  double dt = step_dt(sc);
  sc->dt = dt;
  int p = sc->parity;
  sc->vmax2_bits[p ^ 1] = 0ull;
  sc->parity = p ^ 1;
  sc->n_steps += 1;
  if (dt_trace) dt_trace[sc->trace_pos % trace_ring] = dt;
  sc->trace_pos += 1;
  int r = sc->force_rebuild || (__uint_as_float(sc->maxdisp2_bits) > half_skin2);
  sc->maxdisp2_bits = 0u;  // k_kick_drift of the next step accumulates the displacement since the build again
  sc->do_rebuild = r;
  sc->force_rebuild = 0;
  sc->zbl_count = 0;
  if (r) sc->n_rebuilds += 1;
#if defined(__CUDA_ARCH__)
  if (use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)cond_rebuild, (unsigned)r);
#endif
}

// one thread, after k_force: run the ZBL node of the captured graph only if an atom was flagged
__global__ void k_zbl_gate(const Scalars* sc, unsigned long long cond_zbl) {
  cudaGraphSetConditional((cudaGraphConditionalHandle)cond_zbl, sc->zbl_count > 0 ? 1u : 0u);
}

// first half-kick + drift + wrap + S1 (fixed-point copy into the sorted slot) + displacement since build
__global__ void __launch_bounds__(256)
k_kick_drift(Scalars* sc, const BoxMap* __restrict__ bm, int n, double* __restrict__ pos,
             double* __restrict__ vel, const float* __restrict__ force,
             const int32_t* __restrict__ types, const double* __restrict__ inv_mass,
             const int* __restrict__ inv_perm, int4* __restrict__ xyzt,
             const int4* __restrict__ xyzt_build) {
  __shared__ float sh[32];
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.0f;
  if (i < n) {
    const double dt = step_dt(sc);
    int t = types ? types[i] : 0;
    double im = inv_mass[t];  // 1 / (m * 103.6426965): acceleration in A/fs^2 per eV/A
    unsigned int u[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      size_t k = (size_t)a * n + i;
      double v = vel[k] + 0.5 * dt * ((double)force[k] * im);
      double xx = pos[k] + dt * v;
      if (bm->pbc[a]) xx -= bm->L[a] * floor(xx / bm->L[a]);
      vel[k] = v;
      pos[k] = xx;
      if (!isfinite(xx)) sc->nonfinite = 1;
      u[a] = fix_coord(isfinite(xx) ? xx : 0.0, bm->lo[a], bm->inv_h[a]);
    }
    int s = inv_perm[i];
    int4 b = xyzt_build[s];
    xyzt[s] = make_int4((int)u[0], (int)u[1], (int)u[2], t);
    float dx = (float)((int)u[0] - b.x) * bm->hf[0];
    float dy = (float)((int)u[1] - b.y) * bm->hf[1];
    float dz = (float)((int)u[2] - b.z) * bm->hf[2];
    d2 = dx * dx + dy * dy + dz * dz;
  }
  float m = block_max_128(d2, sh);
  if (threadIdx.x == 0 && m > 0.0f) atomicMax(&sc->maxdisp2_bits, __float_as_uint(m));
}

// second half-kick; leaves max |v|^2 for the next step's dt (integer atomicMax on the bits of a
// non-negative double is order-independent)
__global__ void __launch_bounds__(256)
k_kick(Scalars* sc, int n, double* __restrict__ vel,
       const float* __restrict__ force, const int32_t* __restrict__ types,
       const double* __restrict__ inv_mass, int do_kick) {
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
  if ((threadIdx.x & 31) == 0 && b) atomicMax(&sc->vmax2_bits[sc->parity], b);
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
  for (int b = threadIdx.x; b < nblocks; b += 256) {
    ep += partial[2 * b];
    ek += partial[2 * b + 1];
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
