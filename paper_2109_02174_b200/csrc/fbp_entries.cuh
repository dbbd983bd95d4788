// fbp_entries.cuh -- the back-projector's operands ("entries"), built from a filtered row.
//
// For detector interval j (between bins j and j+1 of the zero-extended row Q~) and its mirror interval
// D-2-j:   mid_a = (Q~[j]+Q~[j+1])/2,  mid_b = (Q~[D-2-j]+Q~[D-1-j])/2,
//          slope_a = Q~[j+1]-Q~[j],    nslope_b = Q~[D-2-j]-Q~[D-1-j].
// Row layout in 16-byte units, index i = j + guard, i in [0, pitch), pitch = D + 2*guard:
//   fp32: one plane   [pitch] of (mid_a, mid_b, slope_a, nslope_b)
//   fp64: two planes  [pitch] of (mid_a, mid_b)  then  [pitch] of (slope_a, nslope_b)
// Entries with j < -1 or j > D-1 are zero guards: out-of-detector reads return 0 without a branch.
// They are written once by fbp_create (the plan's buffer is zero-filled) and by entries_kernel;
// the filter epilogue (fbp_filter3.cuh) writes only j = -1 .. D-1.
#pragma once
#include <cuda_runtime.h>

namespace fbp {

template <typename T> struct EntryPlanes { static constexpr int value = (int)sizeof(T) / 4; };

__device__ __forceinline__ void store_entry(uint4* erow, int /*pitch*/, int i, float ma, float mb, float sa, float sb)
{
    erow[i] = make_uint4(__float_as_uint(ma), __float_as_uint(mb), __float_as_uint(sa), __float_as_uint(sb));
}
__device__ __forceinline__ void store_entry(uint4* erow, int pitch, int i, double ma, double mb, double sa, double sb)
{
    reinterpret_cast<double2*>(erow)[i] = make_double2(ma, mb);
    reinterpret_cast<double2*>(erow)[pitch + i] = make_double2(sa, sb);
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
    uint4* erow = E + (size_t)row * EntryPlanes<T>::value * ent_pitch;
    for (int i = threadIdx.x; i < ent_pitch; i += blockDim.x) {
        T a0 = yz[i + 1], a1 = yz[i + 2];
        T b0 = yz[ent_pitch - 1 - i], b1 = yz[ent_pitch - i];
        if (scaled) { a0 *= m; a1 *= m; b0 *= m; b1 *= m; }
        store_entry(erow, ent_pitch, i, T(0.5) * (a0 + a1), T(0.5) * (b0 + b1), a1 - a0, b0 - b1);
    }
}

}  // namespace fbp
