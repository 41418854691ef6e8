// nep_zbl_energy_sums_static (include/nepzbl.h): the md_energies reduction for callers that must not allocate --
// code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  It is a variant of
// k_energy_partial / k_energy_final (integrate.cuh) whose block partials live in a FILE-SCOPE device array instead of
// the caller's workspace; nothing here calls cudaMalloc, cudaFree or an allocating library routine.
//
// The array is part of the library image: every GPU that loads libnepzbl.so holds its NOALLOC_SCRATCH_BYTES until the
// process exits.  Every call on a device shares it (it keeps the last call's contents; the ticket word that must start
// at zero is cleared before every launch), so two calls that overlap on the same GPU race -- see the header.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "nepzbl.h"

namespace {

constexpr int NOALLOC_BLOCK = 256;
constexpr int NOALLOC_ITEMS = 16;                                   // atoms per thread
constexpr int NOALLOC_CHUNK = NOALLOC_BLOCK * NOALLOC_ITEMS;        // atoms per block = per pair of partial sums
constexpr int NOALLOC_MAX_BLOCKS = (int)(NEPZBL_STATIC_MAX_ATOMS / NOALLOC_CHUNK);
constexpr double AMU_A2_FS2_TO_EV = 103.6426965;                    // nepzbl.h "Units"
static_assert((long long)NOALLOC_MAX_BLOCKS * NOALLOC_CHUNK == NEPZBL_STATIC_MAX_ATOMS, "maximum = whole chunks");

struct NoAllocScratch {
  unsigned int ticket;                     // blocks finished; MUST be zero at launch
  unsigned int pad[63];
  double partial[2 * NOALLOC_MAX_BLOCKS];  // {e_pot, e_kin} per block; rewritten by every call before it is read
};
// 256 B + 128 KiB.  In HOST code this name is a stand-in for the symbol, not a device address: the address a kernel
// can use comes from cudaGetSymbolAddress (scratch_for_current_device below).
static __device__ __align__(256) NoAllocScratch g_noalloc_scratch;

struct MassTable {
  double m[NEPZBL_STATIC_MAX_TYPES];
};

// Each block sums its chunk of atoms in a fixed tree order and stores the pair in the scratch; the block that draws
// the last ticket sums the pairs in index order (again a fixed tree), so the result does not depend on which block
// that is: bit-reproducible, like md_energies.
__global__ void __launch_bounds__(NOALLOC_BLOCK)
k_energy_sums_static(int n, const double* __restrict__ vel, const double* __restrict__ energy,
                     const int32_t* __restrict__ types, int n_types, const MassTable mass,
                     NoAllocScratch* __restrict__ scratch, double* __restrict__ out) {
  __shared__ double sp[NOALLOC_BLOCK], sk[NOALLOC_BLOCK];
  __shared__ bool last;
  double ep = 0.0, ek = 0.0;
  const int base = blockIdx.x * NOALLOC_CHUNK;
#pragma unroll 4
  for (int k = 0; k < NOALLOC_ITEMS; ++k) {
    const int i = base + k * NOALLOC_BLOCK + threadIdx.x;
    if (i < n) {
      const double vx = vel[i], vy = vel[(size_t)n + i], vz = vel[2 * (size_t)n + i];
      int t = types ? types[i] : 0;
      t = min(max(t, 0), n_types - 1);
      ek += 0.5 * mass.m[t] * AMU_A2_FS2_TO_EV * (vx * vx + vy * vy + vz * vz);
      ep += energy[i];
    }
  }
  sp[threadIdx.x] = ep;
  sk[threadIdx.x] = ek;
  __syncthreads();
  for (int o = NOALLOC_BLOCK / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sp[threadIdx.x] += sp[threadIdx.x + o];
      sk[threadIdx.x] += sk[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    scratch->partial[2 * blockIdx.x] = sp[0];
    scratch->partial[2 * blockIdx.x + 1] = sk[0];
    __threadfence();
    last = atomicAdd(&scratch->ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  ep = ek = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += NOALLOC_BLOCK) {
    ep += __ldcg(&scratch->partial[2 * b]);
    ek += __ldcg(&scratch->partial[2 * b + 1]);
  }
  sp[threadIdx.x] = ep;
  sk[threadIdx.x] = ek;
  __syncthreads();
  for (int o = NOALLOC_BLOCK / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sp[threadIdx.x] += sp[threadIdx.x + o];
      sk[threadIdx.x] += sk[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out[0] = sp[0];
    out[1] = sk[0];
    scratch->ticket = 0u;  // left clean for the next call (which clears it again anyway)
  }
}

int report(char* err, size_t err_len, int code, const char* what, const char* detail = "") {
  if (err && err_len) snprintf(err, err_len, "nep_zbl_energy_sums_static: %s%s", what, detail);
  return code;
}

// Device address of the scratch, resolved ONCE PER DEVICE with that device current.
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
NoAllocScratch* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

cudaError_t scratch_for_current_device(int dev, NoAllocScratch** ptr) {
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t ce = cudaGetSymbolAddress(&p, g_noalloc_scratch);  // the CURRENT device's copy of the symbol
    if (ce != cudaSuccess) return ce;
    g_noalloc_ptr[dev] = static_cast<NoAllocScratch*>(p);
  }
  *ptr = g_noalloc_ptr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" int nep_zbl_energy_sums_static(int64_t n_atoms, const double* dev_vel, const double* dev_energy,
                                          const int32_t* dev_types, int32_t n_types, const double* host_mass,
                                          double* dev_out, void* stream, char* host_err, size_t host_err_len) {
  if (host_err && host_err_len) host_err[0] = 0;
  if (n_atoms < 0 || !dev_vel || !dev_energy || !host_mass || !dev_out)
    return report(host_err, host_err_len, NEPZBL_E_INVALID_ARG, "null pointer or negative n_atoms");
  if (n_atoms > NEPZBL_STATIC_MAX_ATOMS) {
    char d[96];
    snprintf(d, sizeof d, " (%lld > %lld)", (long long)n_atoms, (long long)NEPZBL_STATIC_MAX_ATOMS);
    return report(host_err, host_err_len, NEPZBL_E_UNSUPPORTED,
                  "n_atoms beyond NEPZBL_STATIC_MAX_ATOMS, the size the static scratch is laid out for", d);
  }
  if (n_types < 1 || n_types > NEPZBL_STATIC_MAX_TYPES)
    return report(host_err, host_err_len, NEPZBL_E_INVALID_ARG, "n_types outside [1, NEPZBL_STATIC_MAX_TYPES]");
  if (n_types > 1 && !dev_types)
    return report(host_err, host_err_len, NEPZBL_E_INVALID_ARG, "dev_types is required when n_types > 1");
  int dev = -1;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) return report(host_err, host_err_len, NEPZBL_E_CUDA, "cudaGetDevice: ", cudaGetErrorString(ce));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
    return report(host_err, host_err_len, NEPZBL_E_UNSUPPORTED, "device ordinal beyond 63");
  cudaPointerAttributes at{};
  ce = cudaPointerGetAttributes(&at, dev_out);
  if (ce != cudaSuccess || at.type != cudaMemoryTypeDevice || at.device != dev) {
    (void)cudaGetLastError();
    return report(host_err, host_err_len, NEPZBL_E_INVALID_ARG,
                  "dev_out is not device memory of the CURRENT device (make the buffers' device current first)");
  }
  NoAllocScratch* scratch = nullptr;
  ce = scratch_for_current_device(dev, &scratch);
  if (ce != cudaSuccess)
    return report(host_err, host_err_len, NEPZBL_E_CUDA, "cudaGetSymbolAddress: ", cudaGetErrorString(ce));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (n_atoms == 0) {  // nothing to sum: both totals are zero (no launch with an empty grid)
    ce = cudaMemsetAsync(dev_out, 0, 2 * sizeof(double), st);
    if (ce != cudaSuccess) return report(host_err, host_err_len, NEPZBL_E_CUDA, "cudaMemsetAsync: ", cudaGetErrorString(ce));
    return NEPZBL_OK;
  }
  MassTable mt{};
  for (int t = 0; t < n_types; ++t) mt.m[t] = host_mass[t];
  // the ticket must start at zero whatever an earlier (possibly failed) call left behind
  ce = cudaMemsetAsync(&scratch->ticket, 0, sizeof(unsigned int), st);
  if (ce != cudaSuccess) return report(host_err, host_err_len, NEPZBL_E_CUDA, "cudaMemsetAsync: ", cudaGetErrorString(ce));
  const int nb = (int)((n_atoms + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK);
  k_energy_sums_static<<<nb, NOALLOC_BLOCK, 0, st>>>((int)n_atoms, dev_vel, dev_energy, dev_types, n_types, mt, scratch,
                                                     dev_out);
  ce = cudaGetLastError();
  if (ce != cudaSuccess) return report(host_err, host_err_len, NEPZBL_E_CUDA, "launch: ", cudaGetErrorString(ce));
  return NEPZBL_OK;
}
