// nve_kernels.cuh -- the velocity-Verlet integrator of the NVE loop ("velocity-Verlet time
// integration", P:86 NVE) and the two sums its energy needs.  State in fp64 (positions
// [N][3], velocities [N][3], inverse masses [N]); the force kernels read the positions rounded to fp32 from the
// float4 {x, y, z, q} array this kernel keeps in step.  Units: A, e, amu, tau = sqrt(amu A^3 / e^2) (reading Q21).
//
//   v(t + dt/2) = v(t) + (dt/2) F(x(t)) / m;   x(t + dt) = x(t) + dt v(t + dt/2)        nve_kick_kernel, drift on
//   v(t + dt)   = v(t + dt/2) + (dt/2) F(x(t + dt)) / m                                   nve_kick_kernel, drift off
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rbe {

__global__ void __launch_bounds__(256) nve_kick_kernel(double* __restrict__ vel, const double* __restrict__ inv_mass,
                                                        const float4* __restrict__ force, double half_dt, double* __restrict__ pos,
                                                        float4* __restrict__ xyzq, double dt, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 f = force[i];
    const double s = half_dt * inv_mass[i];
    const double vx = fma(s, (double)f.x, vel[3 * i]), vy = fma(s, (double)f.y, vel[3 * i + 1]), vz = fma(s, (double)f.z, vel[3 * i + 2]);
    vel[3 * i] = vx; vel[3 * i + 1] = vy; vel[3 * i + 2] = vz;
    if (pos) {
        const double x = fma(dt, vx, pos[3 * i]), y = fma(dt, vy, pos[3 * i + 1]), z = fma(dt, vz, pos[3 * i + 2]);
        pos[3 * i] = x; pos[3 * i + 1] = y; pos[3 * i + 2] = z;
        float4 a = xyzq[i];
        a.x = (float)x; a.y = (float)y; a.z = (float)z;
        xyzq[i] = a;
    }
}

constexpr int NVE_RED_CTAS = 128;   // per-CTA partials of the two sums below (fixed grid: fixed order)

// partial[b] = sum over this CTA's strided atoms of { 1/2 m v^2, force[i].w }: thread-strided fp64, then a fixed tree
__global__ void __launch_bounds__(256) nve_energy_partial_kernel(const double* __restrict__ vel, const double* __restrict__ inv_mass,
                                                                  const float4* __restrict__ force, int64_t N, double2* __restrict__ partial) {
    __shared__ double2 sh[256];
    double ke = 0.0, sw = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < N; i += (int64_t)gridDim.x * 256) {
        if (vel) {
            const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
            // a frozen atom (inverse mass 0: the kick never moves it) has no finite kinetic energy to report and is
            // left out of the sum; dividing by its inverse mass would turn the whole sum into NaN (0 / 0) or inf
            const double im = inv_mass[i];
            if (im > 0.0) ke += 0.5 * (vx * vx + vy * vy + vz * vz) / im;
        }
        if (force) sw += (double)force[i].w;
    }
    sh[threadIdx.x] = make_double2(ke, sw);
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) { sh[threadIdx.x].x += sh[threadIdx.x + s].x; sh[threadIdx.x].y += sh[threadIdx.x + s].y; }
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(NVE_RED_CTAS) nve_energy_final_kernel(const double2* __restrict__ partial, int n, double* __restrict__ out) {
    __shared__ double2 sh[NVE_RED_CTAS];
    sh[threadIdx.x] = (int)threadIdx.x < n ? partial[threadIdx.x] : make_double2(0.0, 0.0);
    __syncthreads();
    for (int s = NVE_RED_CTAS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) { sh[threadIdx.x].x += sh[threadIdx.x + s].x; sh[threadIdx.x].y += sh[threadIdx.x + s].y; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sh[0].x; out[1] = sh[0].y; }
}

}  // namespace rbe
