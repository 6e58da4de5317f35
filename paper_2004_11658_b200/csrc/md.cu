// md.cu — kernels of the molecular-dynamics driver dpb_md_run (velocity-Verlet,
// NVE).  Units: Angstrom, fs, amu, eV; 1 amu A^2/fs^2 = 103.6426965268 eV (CODATA 2018), k_B = 8.617333262e-5 eV/K.
#include "common.cuh"

// v <- v + (dt/2) F/m;  x <- x + dt v     (hm[t] = (dt/2) / (m_t 103.64...))
__global__ void k_md_kick_drift(int n, double *__restrict__ coord, double *__restrict__ vel,
                                const double *__restrict__ force, const int *__restrict__ type,
                                const double *__restrict__ hm, double dt) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= 3 * n) return;
  const double v = fma(hm[type[k / 3]], force[k], vel[k]);
  vel[k] = v;
  coord[k] = fma(dt, v, coord[k]);
}

// v <- v + (dt/2) F/m
__global__ void k_md_kick(int n, double *__restrict__ vel, const double *__restrict__ force,
                          const int *__restrict__ type, const double *__restrict__ hm) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= 3 * n) return;
  vel[k] = fma(hm[type[k / 3]], force[k], vel[k]);
}

// thermo[slot] = (E_pot, E_kin, T, P [bar]): fixed-order reduction by one block; P = (2 E_kin + tr Xi) / (3 V)
__global__ void k_md_thermo(int n, const double *__restrict__ vel, const int *__restrict__ type,
                            const double *__restrict__ mass_ev, const double *__restrict__ epot,
                            const double *__restrict__ virial, double volume, double *__restrict__ thermo, int slot) {
  __shared__ double part[1024];
  double s = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) {
    const double vx = vel[3 * (size_t)i], vy = vel[3 * (size_t)i + 1], vz = vel[3 * (size_t)i + 2];
    s += 0.5 * mass_ev[type[i]] * (vx * vx + vy * vy + vz * vz);
  }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) part[threadIdx.x] += part[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const double ek = part[0];
    thermo[4 * slot + 0] = *epot;
    thermo[4 * slot + 1] = ek;
    thermo[4 * slot + 2] = n > 0 ? 2.0 * ek / (3.0 * (double)n * 8.617333262e-5) : 0.0;
    thermo[4 * slot + 3] = (2.0 * ek + virial[0] + virial[4] + virial[8]) / (3.0 * volume) * 1.602176634e6;
  }
}

cudaError_t launch_md_kick_drift(int64_t n, double *coord, double *vel, const double *force, const int *type,
                                 const double *hm, double dt, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_md_kick_drift<<<(unsigned)((3 * n + 255) / 256), 256, 0, st>>>((int)n, coord, vel, force, type, hm, dt);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_md_kick(int64_t n, double *vel, const double *force, const int *type, const double *hm,
                           cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_md_kick<<<(unsigned)((3 * n + 255) / 256), 256, 0, st>>>((int)n, vel, force, type, hm);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_md_thermo(int64_t n, const double *vel, const int *type, const double *mass_ev, const double *epot,
                             const double *virial, double volume, double *thermo, int slot, cudaStream_t st) {
  k_md_thermo<<<1, 1024, 0, st>>>((int)n, vel, type, mass_ev, epot, virial, volume, thermo, slot);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// E_kin = sum_i 1/2 m_i v_i^2 of n atoms (eV), fixed-order reduction by one block: the local part of a sub-region, summed
// over the ranks by the decomposition driver (dd.py).
__global__ void k_md_ekin(int n, const double *__restrict__ vel, const int *__restrict__ type,
                          const double *__restrict__ mass_ev, double *__restrict__ ekin) {
  __shared__ double part[1024];
  double s = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) {
    const double vx = vel[3 * (size_t)i], vy = vel[3 * (size_t)i + 1], vz = vel[3 * (size_t)i + 2];
    s += 0.5 * mass_ev[type[i]] * (vx * vx + vy * vy + vz * vz);
  }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) part[threadIdx.x] += part[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) *ekin = part[0];
}

cudaError_t launch_md_ekin(int64_t n, const double *vel, const int *type, const double *mass_ev, double *ekin,
                           cudaStream_t st) {
  k_md_ekin<<<1, 1024, 0, st>>>((int)n, vel, type, mass_ev, ekin);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}
