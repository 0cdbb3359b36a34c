// md_noalloc.cu — md_kinetic_energy_noalloc: the kinetic-energy reduction of md_get_energies (block partials, then one
// fixed-order sum) for callers that may not allocate: its scratch is a file-scope device array of fixed size instead of
// a slice of a workspace.  Not part of the MD path (md_step never calls it) and excluded, like md_probe.cu, from the
// source hash that ties the ncu captures in profiles/ to the kernels they profiled.
//
// E_kin = sum_i 1/2 m_i |v_i|^2 is the first term of the pressure of eq.(6) and the quantity the
// thermostat of eq.(4) acts on.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "md_internal.cuh"

namespace md {

constexpr int kNaThreads = 256, kNaPerThread = 4, kNaAtomsPerBlock = kNaThreads * kNaPerThread;      // 1024 atoms per block
constexpr int kNaMaxBlocks = MD_NOALLOC_MAX_ATOMS / kNaAtomsPerBlock;                               // 4096 partials
constexpr int kNaTicket = kNaMaxBlocks;                        // word index of the arrival counter (offset 32 KB: 256-aligned)
constexpr int kNaWords = kNaMaxBlocks + 32;                    // 33,024 bytes on every device that loads the library
static_assert(MD_NOALLOC_MAX_ATOMS % kNaAtomsPerBlock == 0, "the maximum is a whole number of blocks");

// The scratch: words [0, kNaMaxBlocks) hold one partial sum per block, word kNaTicket counts the blocks that have
// stored theirs (must be 0 when a launch starts; the launch leaves it at 0 and the entry point clears it anyway).
// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address.
static __device__ __align__(256) double g_noalloc_scratch[kNaWords];

struct NaMass { double m[MD_MAX_TYPES]; };

__global__ void __launch_bounds__(kNaThreads) k_ekin_noalloc(const double *__restrict__ v, const int *__restrict__ type,
                                                             const NaMass mp, int n, double *scratch, double *out) {
  __shared__ double sm[kNaThreads / 32];
  __shared__ bool last;
  const int base = blockIdx.x * kNaAtomsPerBlock + threadIdx.x;
  double e = 0.0;
#pragma unroll
  for (int u = 0; u < kNaPerThread; ++u) {
    const int i = base + u * kNaThreads;
    if (i < n) {
      const double vx = v[3 * (size_t)i], vy = v[3 * (size_t)i + 1], vz = v[3 * (size_t)i + 2];
      e += 0.5 * mp.m[type ? type[i] : 0] * (vx * vx + vy * vy + vz * vz);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = e;
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < kNaThreads / 32; ++w) a += sm[w];
    scratch[blockIdx.x] = a;
    __threadfence();                                                       // the partial is visible before the ticket is
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + kNaTicket);
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  // the last block to arrive: all partials of this launch are stored; sum them in an order that depends on nothing
  const volatile double *part = scratch;
  double a = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += kNaThreads) a += part[b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kNaThreads / 32; ++w) t += sm[w];
    *out = t;
    *reinterpret_cast<unsigned *>(scratch + kNaTicket) = 0u;              // ready for the next launch
  }
}

// Device address of the scratch on the CURRENT device: asked for once per device, with that device current.
constexpr int kNaMaxDevices = 64;
static std::mutex g_na_mutex;
static double *g_na_ptr[kNaMaxDevices];

static cudaError_t noalloc_scratch(double **p, int *dev) {
  cudaError_t e = cudaGetDevice(dev);
  if (e != cudaSuccess) return e;
  if (*dev < 0 || *dev >= kNaMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_ptr[*dev]) {
    void *q = nullptr;
    e = cudaGetSymbolAddress(&q, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_na_ptr[*dev] = static_cast<double *>(q);
  }
  *p = g_na_ptr[*dev];
  return cudaSuccess;
}

}  // namespace md

extern "C" int md_kinetic_energy_noalloc(void *stream, const double *v, const int *types, const double *mass, int n_types,
                                         int n_atoms, double *ekin, char *err, int err_len) {
  using namespace md;
  auto fail = [&](int rc, const char *fmt, ...) {
    if (err && err_len > 0) {
      va_list ap;
      va_start(ap, fmt);
      vsnprintf(err, (size_t)err_len, fmt, ap);
      va_end(ap);
    }
    return rc;
  };
  if (err && err_len > 0) err[0] = 0;
  if (n_atoms < 0) return fail(MD_EINVAL, "md_kinetic_energy_noalloc: n_atoms = %d is negative", n_atoms);
  if (n_atoms > MD_NOALLOC_MAX_ATOMS)
    return fail(MD_EINVAL, "md_kinetic_energy_noalloc: n_atoms = %d exceeds MD_NOALLOC_MAX_ATOMS = %d (the fixed scratch array)",
                n_atoms, (int)MD_NOALLOC_MAX_ATOMS);
  if (!ekin || !mass || (n_atoms > 0 && !v)) return fail(MD_EINVAL, "md_kinetic_energy_noalloc: v, mass and ekin must not be NULL");
  if (n_types < 1 || n_types > MD_MAX_TYPES) return fail(MD_EINVAL, "md_kinetic_energy_noalloc: n_types = %d not in 1..%d", n_types, (int)MD_MAX_TYPES);
  if (n_types > 1 && !types && n_atoms > 0) return fail(MD_EINVAL, "md_kinetic_energy_noalloc: types is NULL with n_types = %d", n_types);
  NaMass mp;
  for (int t = 0; t < MD_MAX_TYPES; ++t) {
    if (t < n_types && !(mass[t] > 0.0 && mass[t] < 1e300)) return fail(MD_EINVAL, "md_kinetic_energy_noalloc: mass[%d] is not a positive finite number", t);
    mp.m[t] = t < n_types ? mass[t] * kAmuToEvFs2PerA2 : 0.0;
  }
  double *scratch = nullptr;
  int dev = -1;
  cudaError_t e = noalloc_scratch(&scratch, &dev);
  if (e != cudaSuccess) return fail(MD_ECUDA, "md_kinetic_energy_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
  cudaStream_t st = (cudaStream_t)stream;
  e = cudaMemsetAsync(scratch + kNaTicket, 0, sizeof(double), st);        // the arrival counter starts at zero whatever came before
  if (e != cudaSuccess) return fail(MD_ECUDA, "md_kinetic_energy_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
  const int blocks = n_atoms > 0 ? (n_atoms + kNaAtomsPerBlock - 1) / kNaAtomsPerBlock : 1;
  k_ekin_noalloc<<<blocks, kNaThreads, 0, st>>>(v, n_types > 1 ? types : nullptr, mp, n_atoms, scratch, ekin);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MD_ECUDA, "md_kinetic_energy_noalloc: kernel launch: %s", cudaGetErrorString(e));
  return MD_OK;
}
