// fbp_entries.cuh -- the back-projector's operands ("entries"), built from a filtered row.
//
// One 16-byte unit per detector interval j (between bins j and j+1 of the zero-extended row Q~), index
// i = j + guard, i in [0, pitch), pitch = D + 2*guard.  With a0 = Q~[j], a1 = Q~[j+1] and the mirror interval
// D-2-j: b0 = Q~[D-2-j], b1 = Q~[D-1-j]:
//   fp32: (mid_a, mid_b, slope_a, nslope_b) = ((a0+a1)/2, (b0+b1)/2, a1-a0, b0-b1): ONE LDS.128 feeds a pixel
//         and its point-mirror pixel (value = mid + w slope, w in [-1/2, 1/2]);
//   fp64: (a0, b1) = (Q~[j], Q~[D-1-j]): the NEAR end points of the interval and of its mirror; the far end
//         points are the next unit (a1, b0).  value = near (1-w) + far w, w in [0, 1).  Half the bytes of a
//         (mid, slope) entry in fp64, and a thread that walks along a pixel column keeps `near` in registers and
//         loads only `far` (fbp_backproject.cuh).
// Entries with j < -1 or j > D-1 are zero guards: out-of-detector reads return 0 without a branch.
// They are written once by fbp_create (the plan's buffer is zero-filled) and by entries_kernel;
// the filter epilogues (fbp_filter3.cuh, fbp_fft.cuh) write only j = -1 .. D-1.
#pragma once
#include <cuda_runtime.h>

namespace fbp {

// a0, a1: the interval's end points; b0, b1: the mirror interval's (see the header)
__device__ __forceinline__ void store_entry(uint4* erow, int i, float a0, float a1, float b0, float b1)
{
    erow[i] = make_uint4(__float_as_uint(0.5f * (a0 + a1)), __float_as_uint(0.5f * (b0 + b1)),
                         __float_as_uint(a1 - a0), __float_as_uint(b0 - b1));
}
__device__ __forceinline__ void store_entry(uint4* erow, int i, double a0, double /*a1*/, double /*b0*/, double b1)
{
    reinterpret_cast<double2*>(erow)[i] = make_double2(a0, b1);
}

// Plain filtered rows -> entries (fbp_backproject's first step); the same arithmetic as the filter
// epilogue, so fbp_reconstruct == fbp_backproject(fbp_filter) bit for bit.
// yz[k] = Q~[k - 1 - guard], k in [0, pitch + 2): the row with one extra leading zero and the guards;
// the mirror interval of i then starts at yz[pitch - 1 - i].
// wrow: per-row multipliers (fbp_set_angle_weights: angle weight / (pi/K)) or NULL.
template <typename T>
__global__ void __launch_bounds__(256)
entries_kernel(const T* __restrict__ Q, uint4* __restrict__ E, int n_det, int ent_pitch, int ent_guard,
               const T* __restrict__ wrow, int n_angles)
{
    extern __shared__ __align__(16) unsigned char ent_smem_raw[];
    T* yz = reinterpret_cast<T*>(ent_smem_raw);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the back-projector may start its prologue
    const int row = blockIdx.x;
    const T* q = Q + (size_t)row * n_det;
    for (int k = threadIdx.x; k < ent_pitch + 2; k += blockDim.x) {
        const int n = k - 1 - ent_guard;
        yz[k] = (n >= 0 && n < n_det) ? q[n] : T(0);
    }
    __syncthreads();
    const bool scaled = wrow != nullptr;
    const T m = scaled ? wrow[row % n_angles] : T(1);
    uint4* erow = E + (size_t)row * ent_pitch;
    for (int i = threadIdx.x; i < ent_pitch; i += blockDim.x) {
        T a0 = yz[i + 1], a1 = yz[i + 2];
        T b0 = yz[ent_pitch - 1 - i], b1 = yz[ent_pitch - i];
        if (scaled) { a0 *= m; a1 *= m; b0 *= m; b1 *= m; }
        store_entry(erow, i, a0, a1, b0, b1);
    }
}

}  // namespace fbp
