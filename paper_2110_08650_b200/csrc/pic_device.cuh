// pic_device.cuh — device helpers shared by the step kernels: tile geometry, B-spline shape
// functions, staggered gather, TMA/mbarrier PTX wrappers, split-integer fixed-point adds.
// Definitions: SURVEY.md §8(c) steps 1-6.
#pragma once
#include <cuda.h>

#include "pic_internal.cuh"

namespace {

// ------------------------------------------------------------------ tile geometry
template <int O> struct Geo {
    // E/B tile: node index range per axis for particles in [0,8) (x,y) / [0,4) (z)
    static constexpr int FL = (O == 3) ? 2 : 1;                       // nodes below 0
    static constexpr int FNX = (O == 1) ? 10 : (O == 2) ? 11 : 12;    // nodes used
    static constexpr int FNY = FNX;
    static constexpr int FNZ = FNX - (PIC_SCX - PIC_SCZ);
    static constexpr int FPX = 12;                                    // row pitch (16 B multiple for TMA)
    static constexpr int FCOMP = FPX * FNY * FNZ;                     // floats per component
    // J tile: rho-node range for old positions in [0,8) and new ones in (-1,9)
    static constexpr int JL = (O == 1) ? 1 : 2;
    static constexpr int JNX = (O == 1) ? 11 : 13;
    static constexpr int JNY = JNX;
    static constexpr int JNZ = JNX - (PIC_SCX - PIC_SCZ);
    static constexpr int JCOMP = JNX * JNY * JNZ;
};

// ------------------------------------------------------------------ shape functions
// B-spline weights of degree O at position xr measured from node 0 of the lattice
// (SURVEY.md §8(c) step 1).  Returns the index of the first node with weight w[0].
template <int O> __device__ __forceinline__ int shape(float xr, float (&w)[O + 1])
{
    if (O == 1) {
        float b = floorf(xr);
        float f = xr - b;
        w[0] = 1.0f - f;
        w[1] = f;
        return (int)b;
    } else if (O == 2) {
        float n = floorf(xr + 0.5f);
        float d = xr - n;
        float a = 0.5f - d, c = 0.5f + d;
        w[0] = 0.5f * a * a;
        w[1] = 0.75f - d * d;
        w[2] = 0.5f * c * c;
        return (int)n - 1;
    } else {
        float b = floorf(xr);
        float f = xr - b;
        float g = 1.0f - f;
        float f2 = f * f, f3 = f2 * f;
        const float s = 1.0f / 6.0f;
        w[0] = g * g * g * s;
        w[1] = (3.0f * f3 - 6.0f * f2 + 4.0f) * s;
        w[2] = (-3.0f * f3 + 3.0f * f2 + 3.0f * f + 1.0f) * s;
        w[3] = f3 * s;
        return (int)b - 1;
    }
}

// sm_100a packed FP32: one FFMA2 issues two independent FMAs, d = a * b + c on register pairs.
__device__ __forceinline__ void ffma2(float& d0, float& d1, float a0, float a1, float b0, float b1)
{
    unsigned long long ra, rb, rc;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a0), "f"(a1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b0), "f"(b1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(d0), "f"(d1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(rc) : "l"(ra), "l"(rb));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(rc));
}

// One staggered component: F(X) = sum F[i,j,k] Wx Wy Wz.
// (Pairing rows with packed FMAs was measured: no gain, 2.93 vs 2.89 ms.)
template <int O>
__device__ __forceinline__ float gather1(const float* __restrict__ t, const float (&wx)[O + 1],
                                         const float (&wy)[O + 1], const float (&wz)[O + 1])
{
    using G = Geo<O>;
    float acc = 0.0f;
#pragma unroll
    for (int c = 0; c <= O; ++c) {
        float az = 0.0f;
#pragma unroll
        for (int b = 0; b <= O; ++b) {
            const float* r = t + (c * G::FNY + b) * G::FPX;
            float ay = 0.0f;
#pragma unroll
            for (int a = 0; a <= O; ++a) ay = fmaf(wx[a], r[a], ay);
            az = fmaf(wy[b], ay, az);
        }
        acc = fmaf(wz[c], az, acc);
    }
    return acc;
}

// Place the O+1 weights of a shape evaluation into the W = O+2 wide Esirkepov window
// (off = 0 or 1 = position of w[0] inside the window).
template <int O>
__device__ __forceinline__ void to_window(const float (&w)[O + 1], int off, float (&s)[O + 2])
{
#pragma unroll
    for (int t = 0; t < O + 2; ++t) {
        float lo = (t <= O) ? w[t < O + 1 ? t : O] : 0.0f;      // off == 0
        float hi = (t >= 1) ? w[t - 1 >= 0 ? t - 1 : 0] : 0.0f; // off == 1
        s[t] = off ? hi : lo;
    }
}

__device__ __forceinline__ int wrapi(int i, int n)
{
    if (i < 0) i += n;
    if (i >= n) i -= n;
    return i;
}

// ------------------------------------------------------------------ TMA + mbarrier (PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, unsigned parity)
{
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}

// one 4-D box {x,y,z,component} of the padded field array -> shared memory
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar,
                                            int x, int y, int z, int c)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(c) : "memory");
}

// ------------------------------------------------------------------ fixed-point deposit
// sm_100a has no native shared-memory float add (red.shared.add.f32 compiles to a
// LDS + FADD + ATOMS.CAST.SPIN retry loop); 32-bit integer adds are native (ATOMS.ADD).
// A contribution c (|c| <= cmax <= 2^e) is therefore split exactly into two integers on the
// grid r = 2^(e-33):  c = (hi * 2^15 + lo) * r,  |hi| <= 2^18, |lo| <= 2^14, accumulated in two
// int32 tiles.  Integer sums are associative, so the tile is bit-reproducible; a node overflows
// only beyond 2^13 full-weight contributions (hi) or 2^17 contributions (lo).  DESIGN.md §deposit.
#define PIC_FIX_MAGIC 12582912.0f          // 1.5 * 2^23: adding it rounds to an integer in the mantissa
#define PIC_FIX_MAGIC_BITS 0x4B400000
#define PIC_FIX_LO_BITS 15
#define PIC_FIX_HI_LOG2 18

// 2^(18-e) with |q|max * |w|max * jf <= 2^e: the same value in every CTA and in the convert kernel
__device__ __forceinline__ float fix_scale_of(const PicDev& d, float jf)
{
    int e = 0;
    frexpf(fmaxf(d.qmax * __int_as_float(d.ctr[CTR_WMAX_BITS]) * jf, 1e-30f), &e);
    return ldexpf(1.0f, PIC_FIX_HI_LOG2 - e);
}

__device__ __forceinline__ void fix_add(int* hi, int* lo, int off, float v)
{
    const float t = v + PIC_FIX_MAGIC;                       // |v| <= 2^18: exact integer round(v)
    const float rem = v - (t - PIC_FIX_MAGIC);               // exact, |rem| <= 1/2
    const float t2 = fmaf(rem, (float)(1 << PIC_FIX_LO_BITS), PIC_FIX_MAGIC);
    atomicAdd(hi + off, __float_as_int(t) - PIC_FIX_MAGIC_BITS);
    atomicAdd(lo + off, __float_as_int(t2) - PIC_FIX_MAGIC_BITS);
}

}  // namespace
