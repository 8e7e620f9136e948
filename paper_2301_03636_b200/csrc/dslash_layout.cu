// dslash_layout.cu -- layout module: canonical AoS <-> native (north_star subsystem (1)).
//
// The paper only says the fields are flat one-dimensional arrays; the canonical layout
// is that array with the loop order of PAPER.md:54.  The native SoA layout (dslash_site.cuh) groups sites
// in vectors of 32 consecutive site indices and stores every component of a vector as one contiguous run,
// so a warp's load of one component of 32 consecutive sites is one contiguous 512-byte run and all
// components of a site share one base address.  Pure data movement; bit-exact.
#include "dslash_kernels.cuh"

namespace dslash {

// dir 0: dst[soa(s,u)] = src[s*NU + u]   dir 1: dst[s*NU + u] = src[soa(s,u)]; one thread per (vector, u, lane).
template <typename U>
__global__ void __launch_bounds__(256) transpose_units_kernel(U* __restrict__ dst, const U* __restrict__ src, unsigned V,
                                                              unsigned NU, int dir) {
    const size_t n = (size_t)((V + VL - 1u) / VL) * NU * VL;  // padded SoA size
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned lane = (unsigned)(i & (VL - 1u));
        const size_t vu = i >> VL_LOG2;
        const unsigned u = (unsigned)(vu % NU);
        const unsigned s = (unsigned)(vu / NU) * VL + lane;
        if (s >= V) continue;  // padding of the last vector
        const size_t aos = (size_t)s * NU + u;
        if (dir == 0)
            dst[i] = src[aos];
        else
            dst[aos] = src[i];
    }
}

// Gauge pack.  Canonical: src[(s*4 + mu)*9 + e].  SoA: dst[soa(s, mu*R + e) with 4R components];
// AoS (12-real): dst[(s*4 + mu)*R + e];  e < R.
template <typename U>
__global__ void __launch_bounds__(256) pack_gauge_kernel(U* __restrict__ dst, const U* __restrict__ src, unsigned V, unsigned R,
                                                         int soa) {
    if (soa) {
        const unsigned NU = 4u * R;
        const size_t n = (size_t)((V + VL - 1u) / VL) * NU * VL;
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
            const unsigned lane = (unsigned)(i & (VL - 1u));
            const size_t vu = i >> VL_LOG2;
            const unsigned me = (unsigned)(vu % NU);  // mu*R + e
            const unsigned s = (unsigned)(vu / NU) * VL + lane;
            if (s >= V) continue;
            const unsigned mu = me / R, e = me - mu * R;
            dst[i] = src[((size_t)s * 4u + mu) * 9u + e];
        }
    } else {
        const size_t n = (size_t)V * 4u * R;
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
            const size_t sm = i / R;  // s*4 + mu
            const unsigned e = (unsigned)(i - sm * R);
            dst[i] = src[sm * 9u + e];
        }
    }
}

static unsigned grid_for(size_t n) {
    size_t b = (n + 255) / 256;
    const size_t cap = 148u * 32u;
    return (unsigned)(b < cap ? (b ? b : 1) : cap);
}

cudaError_t launch_convert_spinor(int precision, int layout_base, void* dst, const void* src, unsigned V, int dir,
                                  cudaStream_t stream) {
    const size_t bytes = (size_t)V * 24u * (precision == 0 ? 8u : 4u);
    if (layout_base == LAYOUT_AOS) return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, stream);
    const unsigned NU = precision == 0 ? 12u : 6u;  // 16-byte units per site
    transpose_units_kernel<uint4><<<grid_for((size_t)V * NU), 256, 0, stream>>>(reinterpret_cast<uint4*>(dst),
                                                                                 reinterpret_cast<const uint4*>(src), V, NU, dir);
    return cudaGetLastError();
}

cudaError_t launch_pack_gauge(int precision, int layout_base, int recon, void* dst, const void* src, unsigned V,
                              cudaStream_t stream) {
    const unsigned R = recon == 12 ? 6u : 9u;
    if (layout_base == LAYOUT_AOS && R == 9)
        return cudaMemcpyAsync(dst, src, (size_t)V * 72u * (precision == 0 ? 8u : 4u), cudaMemcpyDeviceToDevice, stream);
    const size_t n = (size_t)V * 4u * (size_t)R;
    if (precision == 0)
        pack_gauge_kernel<uint4><<<grid_for(n), 256, 0, stream>>>(reinterpret_cast<uint4*>(dst),
                                                                  reinterpret_cast<const uint4*>(src), V, R,
                                                                  layout_base == LAYOUT_SOA);
    else
        pack_gauge_kernel<uint2><<<grid_for(n), 256, 0, stream>>>(reinterpret_cast<uint2*>(dst),
                                                                  reinterpret_cast<const uint2*>(src), V, R,
                                                                  layout_base == LAYOUT_SOA);
    return cudaGetLastError();
}

}  // namespace dslash
