// pic_step.cu — the hot path: one CTA per supercell does gather + Boris + move +
// Esirkepov deposit + in-place compaction of stayers; two small kernels finish the
// resort.  Definitions: SURVEY.md §8(c) steps 1-7 (PAPER.md:60-62 names none of them).
//
// Shared memory per CTA: the supercell's E/B tile with shape-order guards
// and a J tile with guards (a4).  fp32 throughout.
#include <cuda.h>
#include <string.h>

#include "pic_internal.cuh"
#include "../../include/pic_b200.h"

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

// One staggered component: F(X) = sum F[i,j,k] Wx Wy Wz.
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

// Esirkepov density decomposition of one component:
// J_a[i,j,k] += fac * sum_{i'<=i} DS_a(i') * [S0_b S0_c + DS_b S0_c/2 + S0_b DS_c/2 + DS_b DS_c/3]
// jt addresses the window's first node; strides sa, sb, sc follow the flow axis a and the
// two transverse axes.  wa/wb/wc: warp-uniform "some lane uses the last window slot of this axis".
template <int O, bool FIX>
__device__ __forceinline__ void deposit1(float* jt, int* jhi, int* jlo, int base, int sa, int sb, int sc, float fac,
                                         bool wa, bool wb, bool wc, bool lane_wa,
                                         const float (&DSa)[O + 2],
                                         const float (&S0b)[O + 2], const float (&DSb)[O + 2],
                                         const float (&S0c)[O + 2], const float (&DSc)[O + 2])
{
    constexpr int W = O + 2;
#pragma unroll
    for (int c = 0; c < W; ++c) {
        if (c == W - 1 && !wc) continue;
        const float c0 = fac * (S0c[c] + 0.5f * DSc[c]);                 // multiplies S0b
        const float c1 = fac * (0.5f * S0c[c] + (1.0f / 3.0f) * DSc[c]); // multiplies DSb
#pragma unroll
        for (int b = 0; b < W; ++b) {
            if (b == W - 1 && !wb) continue;
            const float br = fmaf(S0b[b], c0, DSb[b] * c1);
            float acc = 0.0f;
#pragma unroll
            for (int a = 0; a < W - 1; ++a) {   // the last prefix is sum(DS) = 0: not written
                if (a == W - 2 && !wa) continue;
                acc = fmaf(DSa[a], br, acc);
                // a lane whose own window is narrow has sum_{t<W-1} DS = 0 up to rounding: make it
                // exactly 0, so that the result does not depend on which lanes share its warp
                if (a == W - 2 && !lane_wa) acc = 0.0f;
                const int off = base + a * sa + b * sb + c * sc;
                if (FIX) {
                    fix_add(jhi, jlo, off, acc);   // (predicating zero adds was measured slower: 6.0 vs 6.7e9)
                } else {
                    if (acc != 0.0f) atomicAdd(jt + off, acc);
                }
            }
        }
    }
}

// ------------------------------------------------------------------ the step kernel
template <int O, bool FIX> constexpr int step_smem_bytes()
{
    return (6 * Geo<O>::FCOMP + (FIX ? 6 : 3) * Geo<O>::JCOMP) * 4;
}

template <int O, bool TMA, bool FIX>
__global__ void __launch_bounds__(PIC_FRAME) pic_step_kernel(const PicDev d, const __grid_constant__ CUtensorMap tmap)
{
    using G = Geo<O>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sF = reinterpret_cast<float*>(smem_raw);                 // E/B tile [6][FNZ][FNY][FPX]
    float* sJ = sF + 6 * G::FCOMP;                                  // float J tile [3][JNZ][JNY][JNX]
    int* sJhi = reinterpret_cast<int*>(sJ);                         // or the fixed-point pair
    int* sJlo = sJhi + 3 * G::JCOMP;
    __shared__ int s_wstay[PIC_FRAME / 32];
    __shared__ int s_wleave[PIC_FRAME / 32];
    __shared__ int s_xbase;
    __shared__ __align__(8) uint64_t s_bar;

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int s = blockIdx.x;
    const int ssx = s % d.nsx, ssy = (s / d.nsx) % d.nsy, ssz = s / (d.nsx * d.nsy);
    const int ox = ssx * PIC_SCX, oy = ssy * PIC_SCY, oz = ssz * PIC_SCZ;
    constexpr int NJ = (FIX ? 6 : 3) * G::JCOMP;

    // ---- a2: stage the E/B tile and clear the J tile
    if (TMA) {
        // one bulk-tensor copy of the whole {12, FNY, FNZ, 6} box from the padded array
        // (periodic halos pre-filled by pic_set_fields); completion on an mbarrier
        if (tid == 0) {
            mbar_init(&s_bar, 1);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&s_bar, 6u * G::FCOMP * sizeof(float));
            tma_load_4d(sF, &tmap, &s_bar, ox /* pad_lo_x == FL: 16 B aligned */, oy + PIC_PAD_LO - G::FL,
                        oz + PIC_PAD_LO - G::FL, 0);
        }
        for (int e = tid; e < NJ; e += PIC_FRAME) sJhi[e] = 0;
        __syncthreads();               // the barrier's init is visible to every waiter
        unsigned spins = 0;
        while (!mbar_try_wait(&s_bar, 0)) {
            if (++spins > (1u << 20)) {   // never hang the GPU on a lost copy
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_TMA_TIMEOUT);
                break;
            }
        }
    } else {
        // plain loads with periodic wrap
        const size_t ncell = (size_t)d.nx * d.ny * d.nz;
        for (int e = tid; e < 6 * G::FNZ * G::FNY * G::FNX; e += PIC_FRAME) {
            int i = e % G::FNX;
            int r = e / G::FNX;
            int j = r % G::FNY;
            r /= G::FNY;
            int k = r % G::FNZ;
            int c = r / G::FNZ;
            int gi = wrapi(ox + i - G::FL, d.nx), gj = wrapi(oy + j - G::FL, d.ny),
                gk = wrapi(oz + k - G::FL, d.nz);
            sF[c * G::FCOMP + (k * G::FNY + j) * G::FPX + i] =
                __ldg(d.F + c * ncell + (size_t)gi + (size_t)d.nx * ((size_t)gj + (size_t)d.ny * gk));
        }
        for (int e = tid; e < NJ; e += PIC_FRAME) sJhi[e] = 0;
    }
    __syncthreads();

    // fixed-point scale per component: 2^(18-e) with |q| wmax jf_a <= 2^e
    float fix_scale[3] = {1.0f, 1.0f, 1.0f};
    if (FIX) {
        fix_scale[0] = fix_scale_of(d, d.jfx);
        fix_scale[1] = fix_scale_of(d, d.jfy);
        fix_scale[2] = fix_scale_of(d, d.jfz);
    }

    const int count = d.sc_count[s];
    const int* tbl = d.tbl_pool + d.tbl_off[s];
    int write_pos = 0;

    for (int base = 0; base < count; base += PIC_FRAME) {
        const int slot = base + tid;
        const bool active = slot < count;
        bool stay = false;
        // lanes past the end of a partly filled warp are ghosts of zero weight
        float4 P = make_float4(0.5f, 0.5f, 0.5f, 0.0f), M = make_float4(0.f, 0.f, 0.f, 0.f);
        uint32_t id = 0;
        int dst = s;
        if (base + warp * 32 < count) {        // warp-uniform: the warp holds at least one particle
            if (active) {
                const size_t idx = (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
                P = d.pos[idx];
                M = d.mom[idx];
                id = d.pid[idx];
            }
            const uint32_t bits = __float_as_uint(M.w);
            const int lc = bits & 0xffff, sp = (bits >> 16) & 0xff;
            const int cx = lc & 7, cy = (lc >> 3) & 7, cz = lc >> 6;

            // ---- a2: gather at x^n
            float E[3], B[3];
            {
                float wu[3][O + 1], ws[3][O + 1];
                int bu[3], bs[3];
                const float f[3] = {P.x, P.y, P.z};
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    bu[a] = shape<O>(f[a], wu[a]);
                    bs[a] = shape<O>(f[a] - 0.5f, ws[a]);
                }
                const int ux_ = cx + bu[0] + G::FL, sx_ = cx + bs[0] + G::FL;
                const int uy_ = (cy + bu[1] + G::FL) * G::FPX, sy_ = (cy + bs[1] + G::FL) * G::FPX;
                const int uz_ = (cz + bu[2] + G::FL) * G::FPX * G::FNY, sz_ = (cz + bs[2] + G::FL) * G::FPX * G::FNY;
                E[0] = gather1<O>(sF + 0 * G::FCOMP + sx_ + uy_ + uz_, ws[0], wu[1], wu[2]);
                E[1] = gather1<O>(sF + 1 * G::FCOMP + ux_ + sy_ + uz_, wu[0], ws[1], wu[2]);
                E[2] = gather1<O>(sF + 2 * G::FCOMP + ux_ + uy_ + sz_, wu[0], wu[1], ws[2]);
                B[0] = gather1<O>(sF + 3 * G::FCOMP + ux_ + sy_ + sz_, wu[0], ws[1], ws[2]);
                B[1] = gather1<O>(sF + 4 * G::FCOMP + sx_ + uy_ + sz_, ws[0], wu[1], ws[2]);
                B[2] = gather1<O>(sF + 5 * G::FCOMP + sx_ + sy_ + uz_, ws[0], ws[1], wu[2]);
            }

            // ---- a3: Boris push and move (step 5)
            const float h = d.h[sp];
            const float umx = fmaf(h, E[0], M.x), umy = fmaf(h, E[1], M.y), umz = fmaf(h, E[2], M.z);
            const float igm = rsqrtf(1.0f + umx * umx + umy * umy + umz * umz);
            const float tx = h * B[0] * igm, ty = h * B[1] * igm, tz = h * B[2] * igm;
            const float sfac = 2.0f / (1.0f + tx * tx + ty * ty + tz * tz);
            const float upx = umx + (umy * tz - umz * ty);
            const float upy = umy + (umz * tx - umx * tz);
            const float upz = umz + (umx * ty - umy * tx);
            const float sx2 = tx * sfac, sy2 = ty * sfac, sz2 = tz * sfac;
            const float unx = fmaf(h, E[0], umx + (upy * sz2 - upz * sy2));
            const float uny = fmaf(h, E[1], umy + (upz * sx2 - upx * sz2));
            const float unz = fmaf(h, E[2], umz + (upx * sy2 - upy * sx2));
            const float ig = rsqrtf(1.0f + unx * unx + uny * uny + unz * unz);
            const float del[3] = {unx * ig * d.dtdx, uny * ig * d.dtdy, unz * ig * d.dtdz};
            M.x = unx; M.y = uny; M.z = unz;

            // new in-cell fraction and cell shift (reading S19)
            const float f0[3] = {P.x, P.y, P.z};
            float fn[3], x1[3];
            int sh[3];
            bool far = false;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                float fp = f0[a] + del[a];
                float fl = floorf(fp);
                float g = fp - fl;
                int shift = (int)fl;
                if (g >= 1.0f) {            // tiny negative fp: fp + 1 rounded up to 1
                    g = 0.0f;
                    shift += 1;
                }
                far |= (shift < -1) | (shift > 1);
                fn[a] = g;
                sh[a] = shift;
                x1[a] = (float)shift + g;   // new position relative to the OLD cell's origin node
            }
            if (far) atomicOr(d.ctr + CTR_ERROR, PIC_DEV_MOVED_TOO_FAR);

            // ---- a4: Esirkepov deposit into the shared J tile
            {
                float S0[3][O + 2], DS[3][O + 2];
                int lo[3];
                bool wide[3], lwide[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    float w0[O + 1], w1[O + 1], s1[O + 2];
                    int b0 = shape<O>(f0[a], w0);
                    int b1 = shape<O>(x1[a], w1);
                    lo[a] = min(b0, b1);
                    lwide[a] = b0 != b1;                            // this lane uses the last window slot
                    wide[a] = __any_sync(0xffffffffu, lwide[a]);    // ... some lane of the warp does
                    to_window<O>(w0, b0 - lo[a], S0[a]);
                    to_window<O>(w1, b1 - lo[a], s1);
#pragma unroll
                    for (int t = 0; t < O + 2; ++t) DS[a][t] = s1[t] - S0[a][t];
                }
                const float qw = d.q[sp] * P.w;
                constexpr int SX = 1, SY = G::JNX, SZ = G::JNX * G::JNY;
                const int j0 = (cx + lo[0] + G::JL) * SX + (cy + lo[1] + G::JL) * SY + (cz + lo[2] + G::JL) * SZ;
                deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 0 * G::JCOMP, SX, SY, SZ, -qw * d.jfx * fix_scale[0],
                                 wide[0], wide[1], wide[2], lwide[0], DS[0], S0[1], DS[1], S0[2], DS[2]);
                deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 1 * G::JCOMP, SY, SZ, SX, -qw * d.jfy * fix_scale[1],
                                 wide[1], wide[2], wide[0], lwide[1], DS[1], S0[2], DS[2], S0[0], DS[0]);
                deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 2 * G::JCOMP, SZ, SX, SY, -qw * d.jfz * fix_scale[2],
                                 wide[2], wide[0], wide[1], lwide[2], DS[2], S0[0], DS[0], S0[1], DS[1]);
            }

            // ---- a5: new cell and destination supercell
            int ncx = cx + sh[0], ncy = cy + sh[1], ncz = cz + sh[2];
            int dsx = (ncx < 0) ? -1 : (ncx >= PIC_SCX) ? 1 : 0;
            int dsy = (ncy < 0) ? -1 : (ncy >= PIC_SCY) ? 1 : 0;
            int dsz = (ncz < 0) ? -1 : (ncz >= PIC_SCZ) ? 1 : 0;
            ncx -= dsx * PIC_SCX; ncy -= dsy * PIC_SCY; ncz -= dsz * PIC_SCZ;
            stay = active && (dsx | dsy | dsz) == 0;
            if (active && !stay)
                dst = wrapi(ssx + dsx, d.nsx) + d.nsx * (wrapi(ssy + dsy, d.nsy) + d.nsy * wrapi(ssz + dsz, d.nsz));
            P.x = fn[0]; P.y = fn[1]; P.z = fn[2];
            M.w = __uint_as_float(pic_pack_bits(ncx + PIC_SCX * (ncy + PIC_SCY * ncz), sp));
        }

        // ---- a5: stable compaction of stayers, leavers to the exchange buffer
        const bool leave = active && !stay;
        const unsigned mstay = __ballot_sync(0xffffffffu, stay);
        const unsigned mleave = __ballot_sync(0xffffffffu, leave);
        if (lane == 0) {
            s_wstay[warp] = __popc(mstay);
            s_wleave[warp] = __popc(mleave);
        }
        __syncthreads();   // also: every load of this iteration is complete
        int pre_stay = 0, pre_leave = 0, tot_stay = 0, tot_leave = 0;
#pragma unroll
        for (int w = 0; w < PIC_FRAME / 32; ++w) {
            int a = s_wstay[w], b = s_wleave[w];
            if (w < warp) { pre_stay += a; pre_leave += b; }
            tot_stay += a; tot_leave += b;
        }
        if (tot_leave > 0) {        // block-uniform
            if (tid == 0) s_xbase = atomicAdd(d.ctr + CTR_EXCH, tot_leave);
            __syncthreads();
        }
        const unsigned below = (1u << lane) - 1u;
        if (stay) {
            const int ws = write_pos + pre_stay + __popc(mstay & below);
            const size_t idx = (size_t)tbl[ws >> 8] * PIC_FRAME + (ws & (PIC_FRAME - 1));
            d.pos[idx] = P;
            d.mom[idx] = M;
            d.pid[idx] = id;
        } else if (leave) {
            const int xs = s_xbase + pre_leave + __popc(mleave & below);
            if (xs < d.x_cap) {
                d.x_pos[xs] = P;
                d.x_mom[xs] = M;
                d.x_id[xs] = id;
                d.x_dst[xs] = dst;
                atomicAdd(d.sc_incoming + dst, 1);
            } else {
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_EXCHANGE_OVERFLOW);
            }
        }
        write_pos += tot_stay;
        __syncthreads();   // s_w* / s_xbase are rewritten next iteration
    }
    if (tid == 0) d.sc_stay[s] = write_pos;
    __syncthreads();

    // ---- a4: flush the J tile once (periodic wrap on write)
    {
        const size_t ncell = (size_t)d.nx * d.ny * d.nz;
        for (int e = tid; e < 3 * G::JCOMP; e += PIC_FRAME) {
            int i = e % G::JNX;
            int r = e / G::JNX;
            int j = r % G::JNY;
            r /= G::JNY;
            int k = r % G::JNZ;
            int c = r / G::JNZ;
            int gi = wrapi(ox + i - G::JL, d.nx), gj = wrapi(oy + j - G::JL, d.ny),
                gk = wrapi(oz + k - G::JL, d.nz);
            const size_t g = c * ncell + (size_t)gi + (size_t)d.nx * ((size_t)gj + (size_t)d.ny * gk);
            if (FIX) {
                // 64-bit fixed point in global memory too (native RED.64 in L2): J is bit-reproducible
                const long long n = ((long long)sJhi[e] << PIC_FIX_LO_BITS) + (long long)sJlo[e];
                if (n != 0) atomicAdd(reinterpret_cast<unsigned long long*>(d.J64) + g, (unsigned long long)n);
            } else {
                const float v = sJ[e];
                if (v != 0.0f) atomicAdd(d.J + g, v);
            }
        }
    }
}

// Fixed-point global accumulators -> float J (one pass, after every CTA has flushed).
__global__ void pic_convert_J_kernel(const PicDev d)
{
    const size_t ncell = (size_t)d.nx * d.ny * d.nz;
    const float jf[3] = {d.jfx, d.jfy, d.jfz};
    for (int c = 0; c < 3; ++c) {
        const double inv = 1.0 / ((double)fix_scale_of(d, jf[c]) * (double)(1 << PIC_FIX_LO_BITS));
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < ncell; i += (size_t)gridDim.x * blockDim.x)
            d.J[c * ncell + i] = (float)((double)d.J64[c * ncell + i] * inv);
    }
}

// ------------------------------------------------------------------ resort, part 2
// One thread per supercell: make sure the frame list can hold stayers + arrivals.
__global__ void pic_prepare_kernel(const PicDev d)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.nsc) return;
    const int stay = d.sc_stay[s];
    const int inc = d.sc_incoming[s];
    const int need = (stay + inc + PIC_FRAME - 1) / PIC_FRAME;
    int have = d.sc_nframes[s];
    if (need > have) {
        int off = d.tbl_off[s];
        if (need > d.tbl_cap[s]) {           // grow the frame table (old region is abandoned)
            const int ncap = max(2 * d.tbl_cap[s], need + 4);
            const int noff = atomicAdd(d.ctr + CTR_TBL_TOP, ncap);
            if (noff + ncap > d.tbl_pool_size) {
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_TABLE_POOL_EXHAUSTED);
                return;
            }
            for (int i = 0; i < have; ++i) d.tbl_pool[noff + i] = d.tbl_pool[off + i];
            d.tbl_off[s] = off = noff;
            d.tbl_cap[s] = ncap;
        }
        const int nnew = need - have;
        const int f0 = atomicAdd(d.ctr + CTR_POOL_TOP, nnew);
        if (f0 + nnew > d.n_frames) {
            atomicOr(d.ctr + CTR_ERROR, PIC_DEV_FRAME_POOL_EXHAUSTED);
            return;
        }
        for (int i = 0; i < nnew; ++i) d.tbl_pool[off + have + i] = f0 + i;
        d.sc_nframes[s] = need;
    }
    d.sc_count[s] = stay;
    d.sc_incoming[s] = 0;
    atomicMax(d.ctr + CTR_MAX_COUNT, stay + inc);
}

// One thread per leaver: claim a slot at the tail of the destination's frame list.
__global__ void pic_scatter_kernel(const PicDev d)
{
    const int n = min(d.ctr[CTR_EXCH], d.x_cap);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        d.ctr[CTR_LEAVERS_LAST] = n;
        atomicAdd(d.ctr64 + CTR64_LEAVERS_CUM, (unsigned long long)n);
    }
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int dst = d.x_dst[i];
        const int slot = atomicAdd(d.sc_count + dst, 1);
        const int fr = slot >> 8;
        if (fr < d.sc_nframes[dst]) {
            const size_t idx = (size_t)d.tbl_pool[d.tbl_off[dst] + fr] * PIC_FRAME + (slot & (PIC_FRAME - 1));
            d.pos[idx] = d.x_pos[i];
            d.mom[idx] = d.x_mom[i];
            d.pid[idx] = d.x_id[i];
        }
    }
}

}  // namespace

template <int O, bool TMA, bool FIX>
static cudaError_t launch_step_variant(const PicDev& d, const CUtensorMap& map, cudaStream_t st)
{
    static bool configured = false;     // opt in to > 48 KB of dynamic shared memory once
    constexpr int bytes = step_smem_bytes<O, FIX>();
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(pic_step_kernel<O, TMA, FIX>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    pic_step_kernel<O, TMA, FIX><<<d.nsc, PIC_FRAME, bytes, st>>>(d, map);
    return cudaGetLastError();
}

cudaError_t pic_launch_step(const PicDev& d, int order, bool use_tma, bool fixed_point, const void* tmap,
                            cudaStream_t st, int64_t* launches)
{
    CUtensorMap map;
    if (use_tma) memcpy(&map, tmap, sizeof map); else memset(&map, 0, sizeof map);
    cudaError_t e;
#define PIC_GO(O)                                                                               \
    e = use_tma ? (fixed_point ? launch_step_variant<O, true, true>(d, map, st)                 \
                               : launch_step_variant<O, true, false>(d, map, st))               \
                : (fixed_point ? launch_step_variant<O, false, true>(d, map, st)                \
                               : launch_step_variant<O, false, false>(d, map, st))
    switch (order) {
        case 1: PIC_GO(1); break;
        case 2: PIC_GO(2); break;
        default: PIC_GO(3); break;
    }
#undef PIC_GO
    ++*launches;
    if (e == cudaSuccess && fixed_point) {
        pic_convert_J_kernel<<<148 * 8, 256, 0, st>>>(d);
        ++*launches;
        e = cudaGetLastError();
    }
    return e;
}

cudaError_t pic_launch_resort(const PicDev& d, cudaStream_t st, int64_t* launches, bool scatter)
{
    pic_prepare_kernel<<<(d.nsc + 255) / 256, 256, 0, st>>>(d);
    ++*launches;
    if (scatter) {
        pic_scatter_kernel<<<148 * 4, 256, 0, st>>>(d);
        ++*launches;
    }
    return cudaGetLastError();
}
