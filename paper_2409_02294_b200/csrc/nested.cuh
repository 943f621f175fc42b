// nested.cuh -- kernels of row NEXT-3: the coupling between nested 3-D mesh levels, "each
// nested mesh was allocated one GPU" (Fig. 8 :306).  The per-level solve is the single-level convolution
// of cartesian.cuh; what is new here are the element-wise steps at the level boundaries (readings M1-M6 of DESIGN.md
// section 3; the paper prints no coupling scheme and its ref. [13] is not available):
//   M2  restriction  fine -> coarse: mean of the 2 x 2 x 2 children, written over the parent's central (n/2)^3 cells
//   M3  mask         the level's density with those central cells set to zero (the mass outside the child's box)
//   M5  pack         (out_l + E_l) on the parent cells [n/4 - 1, 3n/4]^3 that cross the level boundary, (n/2 + 2)^3 values
//   M5  prolongation trilinear interpolation of the packed parent values onto the child's cell centres, which sit at
//                    parent coordinate n/4 + (2 i - 1)/4: weights 1/4, 3/4 (even i) or 3/4, 1/4 (odd i);  M6: Phi = own + E
// All arrays [z][y][x], x fastest, fp64.  Each kernel is one pass over its output: HBM-bound, coalesced in x, and two
// to three orders of magnitude cheaper than the solves they sit between.
#pragma once
#include <cuda_runtime.h>

namespace pgk {

__global__ void nest_restrict_kernel(const double *__restrict__ fine, double *__restrict__ mean, const int n)
{
    const int q = n / 2;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)q * q * q) return;
    const int x = (int)(idx % q), y = (int)((idx / q) % q), z = (int)(idx / ((long)q * q));
    double s = 0.0;
#pragma unroll
    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
        for (int dy = 0; dy < 2; ++dy) {
            const double2 v = *reinterpret_cast<const double2 *>(fine + ((long)(2 * z + dz) * n + (2 * y + dy)) * n + 2 * x);
            s += v.x;
            s += v.y;
        }
    mean[idx] = s * 0.125;
}

__global__ void nest_absorb_kernel(double *__restrict__ coarse, const double *__restrict__ mean, const int n)
{
    const int q = n / 2, o = n / 4;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)q * q * q) return;
    const int x = (int)(idx % q), y = (int)((idx / q) % q), z = (int)(idx / ((long)q * q));
    coarse[((long)(o + z) * n + (o + y)) * n + (o + x)] = mean[idx];
}

__global__ void nest_mask_kernel(const double *__restrict__ rho, double *__restrict__ out, const int n)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)n * n * n) return;
    const int x = (int)(idx % n), y = (int)((idx / n) % n), z = (int)(idx / ((long)n * n));
    const int lo = n / 4, hi = 3 * (n / 4);
    const bool inside = x >= lo && x < hi && y >= lo && y < hi && z >= lo && z < hi;
    out[idx] = inside ? 0.0 : rho[idx];
}

// halo[J] = out[parent] + (ext ? ext[parent] : 0),  parent = J + n/4 - 1 per axis
__global__ void nest_pack_kernel(const double *__restrict__ out, const double *__restrict__ ext, double *__restrict__ halo,
                                 const int n)
{
    const int m = n / 2 + 2, o = n / 4 - 1;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)m * m * m) return;
    const int x = (int)(idx % m), y = (int)((idx / m) % m), z = (int)(idx / ((long)m * m));
    const long src = ((long)(o + z) * n + (o + y)) * n + (o + x);
    halo[idx] = out[src] + (ext != nullptr ? ext[src] : 0.0);
}

// E[i] = trilinear(halo), Phi[i] = own[i] + E[i];  halo == nullptr (level 0): E = 0
__global__ void nest_prolong_kernel(const double *__restrict__ halo, const double *__restrict__ own, double *__restrict__ ext,
                                    double *__restrict__ phi, const int n)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)n * n * n) return;
    double e = 0.0;
    if (halo != nullptr) {
        const int m = n / 2 + 2;
        const int x = (int)(idx % n), y = (int)((idx / n) % n), z = (int)(idx / ((long)n * n));
        // lower parent (halo index) and its weight: even i = 2k -> k, 1/4; odd i = 2k + 1 -> k + 1, 3/4
        const int jx = (x >> 1) + (x & 1), jy = (y >> 1) + (y & 1), jz = (z >> 1) + (z & 1);
        const double wx = (x & 1) ? 0.75 : 0.25, wy = (y & 1) ? 0.75 : 0.25, wz = (z & 1) ? 0.75 : 0.25;
#pragma unroll
        for (int az = 0; az < 2; ++az)
#pragma unroll
            for (int ay = 0; ay < 2; ++ay)
#pragma unroll
                for (int ax = 0; ax < 2; ++ax) {
                    const double w = ((az ? 1.0 - wz : wz) * (ay ? 1.0 - wy : wy)) * (ax ? 1.0 - wx : wx);
                    e += w * halo[((long)(jz + az) * m + (jy + ay)) * m + (jx + ax)];
                }
    }
    ext[idx] = e;
    phi[idx] = own[idx] + e;
}

}  // namespace pgk
