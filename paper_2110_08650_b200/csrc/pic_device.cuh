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
    if (O == 0) {                        // nearest grid point (the staggered axes of the energy-conserving CIC gather)
        w[0] = 1.0f;
        return (int)floorf(xr + 0.5f);
    } else if (O == 1) {
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

typedef unsigned long long f32x2;      // two floats in one 64-bit register pair
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
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

// ---- per-cell stencil windows (two-phase gather) -----------------------------------------------
// For every particle of one cell the nodes a component needs along one axis lie in a fixed window:
// O+1 nodes where the first node does not depend on the particle (CIC unstaggered, TSC staggered, PQS
// unstaggered), O+2 nodes where it can take two values (the other three cases; the unused node gets weight 0).
template <int O, bool ST> struct AxisWin {
    static constexpr bool JIT = (O & 1) ? ST : !ST;          // first node depends on the particle
    static constexpr int W = JIT ? O + 2 : O + 1;            // nodes in the window
    static constexpr int LOW = (O == 1) ? (ST ? -1 : 0) : (O == 2) ? -1 : (ST ? -2 : -1);   // first node, cell-relative
};

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

// weights of the window AxisWin<O,ST> for in-cell fraction f
template <int O, bool ST>
__device__ __forceinline__ void axis_weights(float f, float (&w)[AxisWin<O, ST>::W])
{
    float w0[O + 1];
    const int b = shape<O>(ST ? f - 0.5f : f, w0);
    if (AxisWin<O, ST>::JIT) {
        float s[O + 2];
        to_window<O>(w0, b - AxisWin<O, ST>::LOW, s);
#pragma unroll
        for (int t = 0; t < AxisWin<O, ST>::W; ++t) w[t] = s[t];
    } else {
#pragma unroll
        for (int t = 0; t < AxisWin<O, ST>::W; ++t) w[t] = w0[t < O + 1 ? t : O];
    }
}

// TSC (the order the metric is quoted on): the same arithmetic as shape<2> + to_window, written without the
// floor / float->int conversions and the per-slot index compares (14 and 7 instructions instead of ~19 each).
// Unstaggered lattice, window nodes -1..2, valid for f in [-0.5, 1.5): nearest node n = (f >= 0.5).
__device__ __forceinline__ void tsc_window4(float f, float (&w)[4])
{
    const bool up = f >= 0.5f;
    const float d = f - (up ? 1.0f : 0.0f);
    const float a = 0.5f - d, c = 0.5f + d;
    const float wa = 0.5f * a * a, wb = 0.75f - d * d, wc = 0.5f * c * c;
    w[0] = up ? 0.0f : wa;
    w[1] = up ? wa : wb;
    w[2] = up ? wb : wc;
    w[3] = up ? wc : 0.0f;
}
template <> __device__ __forceinline__ void axis_weights<2, false>(float f, float (&w)[4]) { tsc_window4(f, w); }
// staggered lattice (nodes at -1/2, 1/2, 3/2): for f in [0,1) the nearest node is always the middle one
template <> __device__ __forceinline__ void axis_weights<2, true>(float f, float (&w)[3])
{
    const float d = f - 0.5f;
    const float a = 0.5f - d, c = 0.5f + d;
    w[0] = 0.5f * a * a;
    w[1] = 0.75f - d * d;
    w[2] = 0.5f * c * c;
}

// both weight sets (unstaggered / staggered lattice) of the three axes for one particle, plain and as
// duplicated pairs {w,w} for the packed FMAs (unused members cost nothing)
template <int O> struct CellWeights {
    float u[3][AxisWin<O, false>::W];
    float s[3][AxisWin<O, true>::W];
    f32x2 u2[3][AxisWin<O, false>::W];
    f32x2 s2[3][AxisWin<O, true>::W];
    __device__ __forceinline__ void set(float fx, float fy, float fz)
    {
        axis_weights<O, false>(fx, u[0]); axis_weights<O, true>(fx, s[0]);
        axis_weights<O, false>(fy, u[1]); axis_weights<O, true>(fy, s[1]);
        axis_weights<O, false>(fz, u[2]); axis_weights<O, true>(fz, s[2]);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int t = 0; t < AxisWin<O, false>::W; ++t) u2[a][t] = pack2(u[a][t], u[a][t]);
#pragma unroll
            for (int t = 0; t < AxisWin<O, true>::W; ++t) s2[a][t] = pack2(s[a][t], s[a][t]);
        }
    }
    template <bool ST> __device__ __forceinline__ float get(int axis, int t) const
    {
        if constexpr (ST) return s[axis][t];
        else return u[axis][t];
    }
    template <bool ST> __device__ __forceinline__ f32x2 get2(int axis, int t) const
    {
        if constexpr (ST) return s2[axis][t];
        else return u2[axis][t];
    }
};

// The nodes of field component C (0..5 = Ex,Ey,Ez,Bx,By,Bz) that the particles of ONE cell can touch,
// held in registers: E_a is staggered along a, B_a along the two other axes.
// The window is stored as register PAIRS of two z planes (PAIR 0; PAIR 2: the odd last plane stays
// scalar) or of two y rows (PAIR 1), so that the x contraction runs as packed fma.rn.f32x2 (SASS FFMA2).
template <int O, int C> struct CellStencil {
    static constexpr bool STX = (C < 3) ? (C == 0) : (C != 3);
    static constexpr bool STY = (C < 3) ? (C == 1) : (C != 4);
    static constexpr bool STZ = (C < 3) ? (C == 2) : (C != 5);
    using WX = AxisWin<O, STX>;
    using WY = AxisWin<O, STY>;
    using WZ = AxisWin<O, STZ>;
    static constexpr int NX = WX::W, NY = WY::W, NZ = WZ::W;
    static constexpr int PAIR = (NZ % 2 == 0) ? 0 : (NY % 2 == 0) ? 1 : 2;
    static constexpr int NZP = NZ / 2, NYP = NY / 2;
    f32x2 Pz[NZP][NY][NX];      // PAIR 0, 2: planes (2k, 2k+1)
    float Lz[NY][NX];           // PAIR 2: last plane
    f32x2 Py[NZ][NYP][NX];      // PAIR 1: rows (2k, 2k+1)

    __device__ __forceinline__ void load(const float* __restrict__ sF, int cx, int cy, int cz)
    {
        using G = Geo<O>;
        const float* t = sF + C * G::FCOMP + (cx + WX::LOW + G::FL) + (cy + WY::LOW + G::FL) * G::FPX +
                         (cz + WZ::LOW + G::FL) * G::FPX * G::FNY;
        float R[NZ][NY][NX];
#pragma unroll
        for (int c = 0; c < NZ; ++c)
#pragma unroll
            for (int b = 0; b < NY; ++b)
#pragma unroll
                for (int a = 0; a < NX; ++a) R[c][b][a] = t[(c * G::FNY + b) * G::FPX + a];
        if constexpr (PAIR == 1) {
#pragma unroll
            for (int c = 0; c < NZ; ++c)
#pragma unroll
                for (int b = 0; b < NYP; ++b)
#pragma unroll
                    for (int a = 0; a < NX; ++a) Py[c][b][a] = pack2(R[c][2 * b][a], R[c][2 * b + 1][a]);
        } else {
#pragma unroll
            for (int c = 0; c < NZP; ++c)
#pragma unroll
                for (int b = 0; b < NY; ++b)
#pragma unroll
                    for (int a = 0; a < NX; ++a) Pz[c][b][a] = pack2(R[2 * c][b][a], R[2 * c + 1][b][a]);
            if constexpr (PAIR == 2) {
#pragma unroll
                for (int b = 0; b < NY; ++b)
#pragma unroll
                    for (int a = 0; a < NX; ++a) Lz[b][a] = R[NZ - 1][b][a];
            }
        }
    }

    // F(X) = sum F[i,j,k] Wx Wy Wz over the window (weights outside the particle's own O+1 nodes are 0)
    __device__ __forceinline__ float eval(const CellWeights<O>& w) const
    {
        float acc = 0.0f;
        if constexpr (PAIR == 1) {
#pragma unroll
            for (int c = 0; c < NZ; ++c) {
                float az = 0.0f;
#pragma unroll
                for (int b = 0; b < NYP; ++b) {
                    f32x2 ay = mul2(w.template get2<STX>(0, 0), Py[c][b][0]);
#pragma unroll
                    for (int a = 1; a < NX; ++a) ay = fma2(w.template get2<STX>(0, a), Py[c][b][a], ay);
                    float y0, y1;
                    unpack2(ay, y0, y1);
                    az = fmaf(w.template get<STY>(1, 2 * b), y0, az);
                    az = fmaf(w.template get<STY>(1, 2 * b + 1), y1, az);
                }
                acc = fmaf(w.template get<STZ>(2, c), az, acc);
            }
        } else {
#pragma unroll
            for (int c = 0; c < NZP; ++c) {
                f32x2 az = 0;
#pragma unroll
                for (int b = 0; b < NY; ++b) {
                    f32x2 ay = mul2(w.template get2<STX>(0, 0), Pz[c][b][0]);
#pragma unroll
                    for (int a = 1; a < NX; ++a) ay = fma2(w.template get2<STX>(0, a), Pz[c][b][a], ay);
                    az = (b == 0) ? mul2(w.template get2<STY>(1, 0), ay) : fma2(w.template get2<STY>(1, b), ay, az);
                }
                float z0, z1;
                unpack2(az, z0, z1);
                acc = fmaf(w.template get<STZ>(2, 2 * c), z0, acc);
                acc = fmaf(w.template get<STZ>(2, 2 * c + 1), z1, acc);
            }
            if constexpr (PAIR == 2) {
                float az = 0.0f;
#pragma unroll
                for (int b = 0; b < NY; ++b) {
                    float ay = 0.0f;
#pragma unroll
                    for (int a = 0; a < NX; ++a) ay = fmaf(w.template get<STX>(0, a), Lz[b][a], ay);
                    az = fmaf(w.template get<STY>(1, b), ay, az);
                }
                acc = fmaf(w.template get<STZ>(2, NZ - 1), az, acc);
            }
        }
        return acc;
    }
};

// 16-byte asynchronous copy global -> shared (LDGSTS), bypassing L1 and the register file
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem)
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

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
// A value v that is a sum of at most 256 contributions |c| <= cmax <= 2^e is therefore scaled by
// 2^(14-e) (|v'| <= 2^22: the magic add below is exact) and split exactly into two integers on the
// grid r = 2^(e-31):  v = (hi * 2^17 + lo) * r,  |hi| <= 2^22, |lo| <= 2^16, accumulated in two
// int32 tiles.  Integer sums are associative, so the tile is bit-reproducible; a node overflows
// only beyond 2^17 full-weight contributions (hi) or 2^15 flushes (lo).  Every caller flushes its
// register sums at least every 256 particles (PIC_FLUSH_MAX), which is what keeps |v'| <= 2^22.
// DESIGN.md §deposit.
#define PIC_FIX_MAGIC 12582912.0f          // 1.5 * 2^23: adding it rounds to an integer in the mantissa
#define PIC_FIX_MAGIC_BITS 0x4B400000
#define PIC_FIX_LO_BITS 17
#define PIC_FIX_HI_LOG2 14
#define PIC_FLUSH_MAX 256                  // particles summed in registers before a flush, at most

// 2^(14-e) with |q|max * |w|max * jf <= 2^e: the same value in every CTA and in the convert kernel
__device__ __forceinline__ float fix_scale_of(const PicDev& d, float jf)
{
    int e = 0;
    frexpf(fmaxf(d.qmax * __int_as_float(d.ctr[CTR_WMAX_BITS]) * jf, 1e-30f), &e);
    return ldexpf(1.0f, PIC_FIX_HI_LOG2 - e);
}

__device__ __forceinline__ void fix_add(int* hi, int* lo, int off, float v)
{
    const float t = v + PIC_FIX_MAGIC;                       // |v| <= 2^22: exact integer round(v)
    const float rem = v - (t - PIC_FIX_MAGIC);               // exact, |rem| <= 1/2
    const float t2 = fmaf(rem, (float)(1 << PIC_FIX_LO_BITS), PIC_FIX_MAGIC);
    atomicAdd(hi + off, __float_as_int(t) - PIC_FIX_MAGIC_BITS);
    atomicAdd(lo + off, __float_as_int(t2) - PIC_FIX_MAGIC_BITS);
}

// two contributions at once: the float part of the split runs as packed f32x2 operations
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ void fix_add2(int* hi, int* lo, int off0, int off1, float v0, float v1)
{
    const f32x2 magic = pack2(PIC_FIX_MAGIC, PIC_FIX_MAGIC), nmagic = pack2(-PIC_FIX_MAGIC, -PIC_FIX_MAGIC);
    const f32x2 v = pack2(v0, v1);
    const f32x2 t = add2(v, magic);                                   // exact integers round(v)
    const f32x2 nr = add2(add2(t, nmagic), pack2(-v0, -v1));          // -(v - round(v)), exact
    const f32x2 t2 = fma2(nr, pack2(-(float)(1 << PIC_FIX_LO_BITS), -(float)(1 << PIC_FIX_LO_BITS)), magic);
    float ta, tb, ua, ub;
    unpack2(t, ta, tb);
    unpack2(t2, ua, ub);
    atomicAdd(hi + off0, __float_as_int(ta) - PIC_FIX_MAGIC_BITS);
    atomicAdd(lo + off0, __float_as_int(ua) - PIC_FIX_MAGIC_BITS);
    atomicAdd(hi + off1, __float_as_int(tb) - PIC_FIX_MAGIC_BITS);
    atomicAdd(lo + off1, __float_as_int(ub) - PIC_FIX_MAGIC_BITS);
}

}  // namespace
