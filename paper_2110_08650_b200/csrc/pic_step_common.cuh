// pic_step_common.cuh — device code shared by the step kernels of pic_step.cu (first and second generation:
// one-phase, two-phase, sparse) and pic_cell.cu (third generation, whole-cell items): Esirkepov straight
// into the shared tile, Boris push + move, write-back / leaver staging, the counting sort fused into the
// prologue.  Definitions: SURVEY.md §8(c) steps 1-7.
#pragma once
#include <cuda.h>

#include "pic_internal.cuh"
#include "pic_device.cuh"
#include "../../include/pic_b200.h"

namespace {

#define PIC_XSTAGE 128     // leavers staged in shared memory per CTA before one bulk append
#define PIC_SLOWCAP_OF(O) ((O) == 3 ? 256 : 32)   // queued out-of-window particles per CTA (then: overflow queue)
#define PIC_STEP_THREADS 128   // 2 CTAs of 4 warps per SM: ~250 registers per thread for the accumulators

// Esirkepov density decomposition of one component, straight into the
// shared tile, with a per-particle window [lo, lo+O+2):
// J_a[i,j,k] += fac * sum_{i'<=i} DS_a(i') * [S0_b S0_c + DS_b S0_c/2 + S0_b DS_c/2 + DS_b DS_c/3]
// wa/wb/wc: warp-uniform "some lane uses the last window slot of this axis".
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
                if (a == W - 2 && !lane_wa) acc = 0.0f;   // narrow lane: exactly 0, whatever its warp
                const int off = base + a * sa + b * sb + c * sc;
                if (FIX) fix_add(jhi, jlo, off, acc);
                else if (acc != 0.0f) atomicAdd(jt + off, acc);
            }
        }
    }
}

// O+1 weights placed in the cell's fixed 4-node window (nodes -1..2); off = first node + 1.
template <int O> __device__ __forceinline__ void place4(const float (&w)[O + 1], int off, float (&s)[4])
{
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        float v = 0.0f;
#pragma unroll
        for (int o = 0; o <= 3 - O; ++o)
            if (t - o >= 0 && t - o <= O) v = (off == o) ? w[t - o] : v;
        s[t] = v;
    }
}

// One out-of-window particle, straight into the tile (all 32 lanes of the warp take part; lanes
// without a particle pass qw = 0 and f0 = x1 = 0.5).
template <int O, bool FIX>
__device__ __forceinline__ void deposit_direct(const PicDev& d, float* sJ, int* sJhi, int* sJlo, const float (&fix_scale)[3],
                                               const float (&f0)[3], const float (&x1)[3], float qw, int lc)
{
    using G = Geo<O>;
    const int cx = lc & 7, cy = (lc >> 3) & 7, cz = lc >> 6;
    float S0[3][O + 2], DS[3][O + 2];
    int lo[3];
    bool wide[3], lwide[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float w0[O + 1], w1[O + 1], s1[O + 2];
        int b0 = shape<O>(f0[a], w0);
        int b1 = shape<O>(x1[a], w1);
        lo[a] = min(b0, b1);
        lwide[a] = b0 != b1;
        wide[a] = __any_sync(0xffffffffu, lwide[a]);
        to_window<O>(w0, b0 - lo[a], S0[a]);
        to_window<O>(w1, b1 - lo[a], s1);
#pragma unroll
        for (int t = 0; t < O + 2; ++t) DS[a][t] = s1[t] - S0[a][t];
    }
    constexpr int SX = 1, SY = G::JNX, SZ = G::JNX * G::JNY;
    const int j0 = (cx + lo[0] + G::JL) * SX + (cy + lo[1] + G::JL) * SY + (cz + lo[2] + G::JL) * SZ;
    deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 0 * G::JCOMP, SX, SY, SZ, -qw * d.jfx * fix_scale[0],
                     wide[0], wide[1], wide[2], lwide[0], DS[0], S0[1], DS[1], S0[2], DS[2]);
    deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 1 * G::JCOMP, SY, SZ, SX, -qw * d.jfy * fix_scale[1],
                     wide[1], wide[2], wide[0], lwide[1], DS[1], S0[2], DS[2], S0[0], DS[0]);
    deposit1<O, FIX>(sJ, sJhi, sJlo, j0 + 2 * G::JCOMP, SZ, SX, SY, -qw * d.jfz * fix_scale[2],
                     wide[2], wide[0], wide[1], lwide[2], DS[2], S0[0], DS[0], S0[1], DS[1]);
}


// register accumulation of one component over the cell's window:
// A[i][b][c] += fac * (sum_{i'<=i} DS_a(i')) * bracket(b,c),  i = nodes -1,0,1 of the flow axis
__device__ __forceinline__ void accumulate1(float (&A)[3][4][4], float fac, const float (&DSa)[4],
                                            const float (&S0b)[4], const float (&DSb)[4],
                                            const float (&S0c)[4], const float (&DSc)[4])
{
    const float p0 = fac * DSa[0];
    const float p1 = fmaf(fac, DSa[1], p0);
    const float p2 = fmaf(fac, DSa[2], p1);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float c0 = S0c[c] + 0.5f * DSc[c];
        const float c1 = 0.5f * S0c[c] + (1.0f / 3.0f) * DSc[c];
        float br[4];
#pragma unroll
        for (int b = 0; b < 4; b += 2) {
            br[b] = DSb[b] * c1;
            br[b + 1] = DSb[b + 1] * c1;
            ffma2(br[b], br[b + 1], S0b[b], S0b[b + 1], c0, c0);
        }
#pragma unroll
        for (int b = 0; b < 4; ++b) ffma2(A[0][b][c], A[1][b][c], p0, p1, br[b], br[b]);
#pragma unroll
        for (int b = 0; b < 4; b += 2) ffma2(A[2][b][c], A[2][b + 1][c], br[b], br[b + 1], p2, p2);
    }
}

template <bool FIX>
__device__ __forceinline__ void flush1(float* sJ, int* sJhi, int* sJlo, int off, float v)
{
    if (FIX) fix_add(sJhi, sJlo, off, v);
    else if (v != 0.0f) atomicAdd(sJ + off, v);
}
template <bool FIX>
__device__ __forceinline__ void flush2(float* sJ, int* sJhi, int* sJlo, int off0, int off1, float v0, float v1)
{
    if (FIX) fix_add2(sJhi, sJlo, off0, off1, v0, v1);
    else {
        if (v0 != 0.0f) atomicAdd(sJ + off0, v0);
        if (v1 != 0.0f) atomicAdd(sJ + off1, v1);
    }
}

// a2 for one particle: gather E,B at x^n from the shared tile.
// ec = false: momentum-conserving gather (reading S3, the contract's path): order O on every axis.
// ec = true: energy-conserving (Galerkin) gather: order O-1 along the axes a component is staggered
//            on (the O weights are padded with a zero, so the same O+1-wide loops run; the extra node read lies
//            inside the tile: it is a node the order-O window of a neighbouring position would touch).
template <int O>
__device__ __forceinline__ void gather_particle(const float* sF, int cx, int cy, int cz, const float4& P,
                                                float (&E)[3], float (&B)[3], bool ec = false)
{
    using G = Geo<O>;
    {
        float wu[3][O + 1], ws[3][O + 1];
        int bu[3], bs[3];
        const float f[3] = {P.x, P.y, P.z};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            bu[a] = shape<O>(f[a], wu[a]);
            if (ec) {
                float wl[O];
                bs[a] = shape<O - 1>(f[a] - 0.5f, wl);
#pragma unroll
                for (int t = 0; t < O; ++t) ws[a][t] = wl[t];
                ws[a][O] = 0.0f;
            } else {
                bs[a] = shape<O>(f[a] - 0.5f, ws[a]);
            }
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
}

// a3 for one particle: Boris push, move (step 5) and the split of the new
// position into cell shift + in-cell fraction (reading S19).
__device__ __forceinline__ void boris_move(const PicDev& d, int sp, const float4& P, const float4& M,
                                           const float (&E)[3], const float (&B)[3], float (&un)[3], float (&fn)[3],
                                           float (&x1)[3], int (&sh)[3])
{
    const float h = d.h[sp];
    const float umx = fmaf(h, E[0], M.x), umy = fmaf(h, E[1], M.y), umz = fmaf(h, E[2], M.z);
    const float igm = rsqrtf(1.0f + umx * umx + umy * umy + umz * umz);
    const float tx = h * B[0] * igm, ty = h * B[1] * igm, tz = h * B[2] * igm;
    const float sfac = __fdividef(2.0f, 1.0f + tx * tx + ty * ty + tz * tz);   // MUFU.RCP, 2 ulp (reading D4)
    const float upx = umx + (umy * tz - umz * ty);
    const float upy = umy + (umz * tx - umx * tz);
    const float upz = umz + (umx * ty - umy * tx);
    const float sx2 = tx * sfac, sy2 = ty * sfac, sz2 = tz * sfac;
    const float unx = fmaf(h, E[0], umx + (upy * sz2 - upz * sy2));
    const float uny = fmaf(h, E[1], umy + (upz * sx2 - upx * sz2));
    const float unz = fmaf(h, E[2], umz + (upx * sy2 - upy * sx2));
    const float ig = rsqrtf(1.0f + unx * unx + uny * uny + unz * unz);
    const float del[3] = {unx * ig * d.dtdx, uny * ig * d.dtdy, unz * ig * d.dtdz};

    // new in-cell fraction and cell shift (reading S19)
    const float f0[3] = {P.x, P.y, P.z};
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
    un[0] = unx; un[1] = uny; un[2] = unz;
}

// a2 + a3 for one particle, gathering from the shared E/B tile.
template <int O>
__device__ __forceinline__ void push_particle(const PicDev& d, const float* sF, int cx, int cy, int cz, int sp,
                                              const float4& P, const float4& M, float (&un)[3], float (&fn)[3],
                                              float (&x1)[3], int (&sh)[3])
{
    float E[3], B[3];
    gather_particle<O>(sF, cx, cy, cz, P, E, B, d.gather_ec != 0);
    boris_move(d, sp, P, M, E, B, un, fn, x1, sh);
}

// One record = one 32-byte DRAM sector, written back as ONE store (st.global.v8.f32, SASS STG.E.ENL2.256): half the
// store instructions and L1 wavefronts of two 16-byte halves.
__device__ __forceinline__ void store_record256(float4* dst, const float4& P, const float4& M)
{
    asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 :: "l"(dst), "f"(P.x), "f"(P.y), "f"(P.z), "f"(P.w), "f"(M.x), "f"(M.y), "f"(M.z), "f"(M.w) : "memory");
}

__device__ __forceinline__ void load_record256(const float4* src, float4& P, float4& M)
{
    asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(P.x), "=f"(P.y), "=f"(P.z), "=f"(P.w), "=f"(M.x), "=f"(M.y), "=f"(M.z), "=f"(M.w) : "l"(src) : "memory");
}

// a5 for one particle: new local cell and destination supercell; stayers are written back in place
// and counted per new cell, leavers leave a flagged hole and are staged for the exchange buffer.
__device__ __forceinline__ void finish_particle(const PicDev& d, float4* rec, size_t idx, int s, int ssx, int ssy, int ssz,
                                                int cx, int cy, int cz, int sp, float4 P, float4 M,
                                                const float (&un)[3], const float (&fn)[3], const int (&sh)[3],
                                                int* s_hist, int* s_xn, float4* s_xrec, uint32_t* s_xid, int* s_xdst)
{
    const float unx = un[0], uny = un[1], unz = un[2];
    // ---- a5: new cell, destination supercell, write back in place
    int ncx = cx + sh[0], ncy = cy + sh[1], ncz = cz + sh[2];
    const int dsx = (ncx < 0) ? -1 : (ncx >= PIC_SCX) ? 1 : 0;
    const int dsy = (ncy < 0) ? -1 : (ncy >= PIC_SCY) ? 1 : 0;
    const int dsz = (ncz < 0) ? -1 : (ncz >= PIC_SCZ) ? 1 : 0;
    ncx -= dsx * PIC_SCX; ncy -= dsy * PIC_SCY; ncz -= dsz * PIC_SCZ;
    const int nlc = ncx + PIC_SCX * (ncy + PIC_SCY * ncz);
    const uint32_t nbits = pic_pack_bits(nlc, sp);
    P.x = fn[0]; P.y = fn[1]; P.z = fn[2];
    M.x = unx; M.y = uny; M.z = unz;
    if ((dsx | dsy | dsz) == 0) {
        M.w = __uint_as_float(nbits);
        store_record256(rec + 2 * idx, P, M);
        atomicAdd(&s_hist[nlc], 1);
    } else {
        const int dst = wrapi(ssx + dsx, d.nsx) + d.nsx * (wrapi(ssy + dsy, d.nsy) + d.nsy * wrapi(ssz + dsz, d.nsz));
        rec[2 * idx + 1] = make_float4(unx, uny, unz, __uint_as_float(nbits | PIC_LEFT_FLAG));   // hole
        M.w = __uint_as_float(nbits);
        const int k = atomicAdd(s_xn, 1);
        if (k < PIC_XSTAGE) {         // the id (a DRAM miss) is fetched by the bulk append, off the particle loop
            s_xrec[2 * k] = P; s_xrec[2 * k + 1] = M; s_xid[k] = (uint32_t)idx; s_xdst[k] = dst;
        } else {                      // staging full: append directly
            const int xs = atomicAdd(d.ctr + CTR_EXCH, 1);
            if (xs < d.x_cap) {
                d.x_rec[2 * (size_t)xs] = P; d.x_rec[2 * (size_t)xs + 1] = M; d.x_id[xs] = d.pid[d.cur][idx]; d.x_dst[xs] = dst;
            } else {
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_EXCHANGE_OVERFLOW);
            }
        }
        atomicAdd(d.cell_hist + (size_t)dst * 256 + nlc, 1);
        atomicAdd(d.sc_incoming + dst, 1);
    }
}

// A supercell whose particles all left in the previous step (population after the pending sort = 0) is skipped by
// every step kernel; when no stand-alone sort runs for it either (class_all == 2) its published count must still be
// reset, or pic_prepare_kernel would build the next tail on the stale value.  Idempotent; one thread.
__device__ __forceinline__ void retire_empty_supercell(const PicDev& d, int s)
{
    if (d.fused && d.sc_count[s] != 0) d.sc_count[s] = 0;
}

// Barrier over the NT threads that run a block-level routine: the whole CTA (BAR == 0, __syncthreads) or one warp
// group of a warp-specialized kernel (named barrier BAR > 0; the other warps of the CTA do not take part).
template <int BAR, int NT> __device__ __forceinline__ void group_sync()
{
    if constexpr (BAR == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"n"(BAR), "n"(NT) : "memory");
}

// ------------------------------------------------------------------ sort fused into the step kernel's prologue
// Exclusive scan over 256 counts held NT-strided in registers (entry tid*PER + k); two block barriers.
template <int NT, int BAR = 0>
__device__ __forceinline__ void block_excl_scan256(int (&v)[256 / NT], int& total, int* s_w, int tid)
{
    constexpr int PER = 256 / NT, NW = NT / 32;
    const int lane = tid & 31, warp = tid >> 5;
    int sum = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) sum += v[k];
    int inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    group_sync<BAR, NT>();               // s_w may still be read from an earlier scan
    if (lane == 31) s_w[warp] = inc;
    group_sync<BAR, NT>();
    int wb = 0;
    total = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const int x = s_w[w];
        if (w < warp) wb += x;
        total += x;
    }
    int off = wb + inc - sum;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int c = v[k];
        v[k] = off;
        off += c;
    }
}

// The counting sort of pic_sort_kernel for ONE supercell, run by the step CTA before it steps the
// supercell: pool cur^1 (stayers, holes of leavers, appended arrivals) -> pool cur, sorted by cell.
// Leaves the cell ranges in s_off[0..256] (shared), publishes the new count, clears the global histogram,
// returns frames the supercell no longer needs.  s_cur: 256 ints of scratch; s_w: 16 ints of scratch.
#define PIC_SORT_TBL 1024
// STAGE_R > 0: the records are not held in registers but requested with cp.async into `scratch` (STAGE_R records per
// thread and round, 36 bytes each, every thread its own entries): as many loads in flight with a handful of
// registers — for the producer warps of the persistent kernel, which run on 56 registers (spilled batch registers
// serialise the loads: the spill store waits for the load).
template <int NT, int BAR = 0, int U = 4, int STAGE_R = 0>
__device__ __forceinline__ int fused_sort(const PicDev& d, int s, int tid, int* s_off, int* s_cur, int* s_w, int* s_tbl_scr,
                                          unsigned char* scratch = nullptr)
{
    constexpr int PER = 256 / NT;
    // slots in use, never beyond the frames the supercell owns (after a frame-pool fault the tail counts particles
    // that found no slot: the table entries behind sc_nframes are not initialised)
    const int n_scan = min(d.sc_tail[s], d.sc_nframes[s] * PIC_FRAME);
    int v[PER];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        v[k] = d.cell_hist_prev[(size_t)s * 256 + tid * PER + k];
        d.cell_hist_prev[(size_t)s * 256 + tid * PER + k] = 0;
    }
    int total;
    block_excl_scan256<NT, BAR>(v, total, s_w, tid);
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        s_off[tid * PER + k] = v[k];
        s_cur[tid * PER + k] = v[k];
    }
    if (tid == 0) {
        s_off[256] = total;
        d.sc_count[s] = total;
    }
    group_sync<BAR, NT>();
    if (total > n_scan || total != d.sc_next[s]) {      // histogram and records disagree: never write out of bounds
        if (tid == 0) atomicOr(d.ctr + CTR_ERROR, PIC_DEV_SORT_MISMATCH);
        return -1;
    }
    // frame table in shared memory (s_tbl_scr: up to PIC_SORT_TBL entries of scratch), else straight from global
    const int have_frames = d.sc_nframes[s];
    const int* tbl = d.tbl_pool + d.tbl_off[s];
    if (have_frames <= PIC_SORT_TBL) {
        for (int t = tid; t < have_frames; t += NT) s_tbl_scr[t] = tbl[t];
        group_sync<BAR, NT>();
        tbl = s_tbl_scr;
    }
    const float4* src = d.rec[d.cur ^ 1];
    float4* dst = d.rec[d.cur];
    const uint32_t* sid = d.pid[d.cur ^ 1];
    uint32_t* did = d.pid[d.cur];
    if constexpr (STAGE_R > 0) {
        float4* sP = reinterpret_cast<float4*>(scratch);
        float4* sM = sP + STAGE_R * NT;
        uint32_t* sI = reinterpret_cast<uint32_t*>(sM + STAGE_R * NT);
        for (int base = 0; base < n_scan; base += STAGE_R * NT) {
#pragma unroll
            for (int u = 0; u < STAGE_R; ++u) {
                const int slot = base + u * NT + tid;
                if (slot < n_scan) {
                    const size_t i = (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
                    cp_async16(sP + u * NT + tid, src + 2 * i);
                    cp_async16(sM + u * NT + tid, src + 2 * i + 1);
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(sI + u * NT + tid)),
                                 "l"(sid + i) : "memory");
                }
            }
            cp_async_wait_all();
#pragma unroll
            for (int u = 0; u < STAGE_R; ++u) {
                const int slot = base + u * NT + tid;
                if (slot >= n_scan) continue;
                const float4 M = sM[u * NT + tid];
                const uint32_t bits = __float_as_uint(M.w);
                if (bits & PIC_LEFT_FLAG) continue;
                const int r = atomicAdd(&s_cur[bits & 0xff], 1);
                if (r >= total) {
                    atomicOr(d.ctr + CTR_ERROR, PIC_DEV_SORT_MISMATCH);
                    continue;
                }
                const size_t o = (size_t)tbl[r >> 8] * PIC_FRAME + (r & (PIC_FRAME - 1));
                dst[2 * o] = sP[u * NT + tid];
                dst[2 * o + 1] = M;
                did[o] = sI[u * NT + tid];
            }
        }
    } else {
    // U slots per thread and batch; the next batch is loaded while the current one is ranked and stored
    struct Batch {
        float4 P[U], M[U];
        uint32_t id[U];
        bool ok[U];
    };
    auto load = [&](Batch& q, int base) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int slot = base + u * NT + tid;
            q.ok[u] = slot < n_scan;
            if (q.ok[u]) {
                const size_t i = (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
                load_record256(src + 2 * i, q.P[u], q.M[u]);
                q.id[u] = __ldcs(sid + i);
            }
        }
    };
    auto place = [&](const Batch& q) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (!q.ok[u]) continue;
            const uint32_t bits = __float_as_uint(q.M[u].w);
            if (bits & PIC_LEFT_FLAG) continue;
            const int r = atomicAdd(&s_cur[bits & 0xff], 1);
            if (r >= total) {
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_SORT_MISMATCH);
                continue;
            }
            const size_t o = (size_t)tbl[r >> 8] * PIC_FRAME + (r & (PIC_FRAME - 1));
            store_record256(dst + 2 * o, q.P[u], q.M[u]);
            did[o] = q.id[u];
        }
    };
    Batch qa, qb;
    load(qa, 0);
    for (int base = 0; base < n_scan; base += 2 * U * NT) {
        load(qb, base + U * NT);           // (slots >= n_scan: nothing is loaded)
        place(qa);
        load(qa, base + 2 * U * NT);
        place(qb);
    }
    }
    group_sync<BAR, NT>();                   // the sorted records are visible to the whole CTA
    if (tid == 0) {
        const int keep = (total + PIC_FRAME - 1) / PIC_FRAME + 1, have = d.sc_nframes[s];
        if (have > keep) {
            const int at = atomicAdd(d.ctr + CTR_FREE_TOP, have - keep);
            for (int i = keep; i < have; ++i) d.free_stack[at + i - keep] = tbl[i];
            d.sc_nframes[s] = keep;
        }
    }
    return total;
}

// ------------------------------------------------------------------ two-phase gather
// The stencils of the components in MASK for one cell (members outside MASK are never touched and cost nothing).
template <int O, int MASK> struct StencilSet {
    CellStencil<O, 0> c0; CellStencil<O, 1> c1; CellStencil<O, 2> c2;
    CellStencil<O, 3> c3; CellStencil<O, 4> c4; CellStencil<O, 5> c5;
    __device__ __forceinline__ void load(const float* sF, int cx, int cy, int cz)
    {
        if constexpr ((MASK & 1) != 0) c0.load(sF, cx, cy, cz);
        if constexpr ((MASK & 2) != 0) c1.load(sF, cx, cy, cz);
        if constexpr ((MASK & 4) != 0) c2.load(sF, cx, cy, cz);
        if constexpr ((MASK & 8) != 0) c3.load(sF, cx, cy, cz);
        if constexpr ((MASK & 16) != 0) c4.load(sF, cx, cy, cz);
        if constexpr ((MASK & 32) != 0) c5.load(sF, cx, cy, cz);
    }
    template <int C> __device__ __forceinline__ float eval(const CellWeights<O>& w) const
    {
        if constexpr (C == 0) return c0.eval(w);
        else if constexpr (C == 1) return c1.eval(w);
        else if constexpr (C == 2) return c2.eval(w);
        else if constexpr (C == 3) return c3.eval(w);
        else if constexpr (C == 4) return c4.eval(w);
        else return c5.eval(w);
    }
};

// One gather pass over the n particles of the thread's item: the components in MASK, each into its
// staging slot (slot = component index).  stgP/stgF point at the thread's own column.
template <int O, int MASK, int NSLOT, bool WAIT>
__device__ __forceinline__ void gather_pass(const float* sF, int cx, int cy, int cz, int n, const float4* stgP, float* stgF)
{
    constexpr int NT = PIC_STEP_THREADS;
    StencilSet<O, MASK> st;
    st.load(sF, cx, cy, cz);
    if (WAIT) cp_async_wait_all();      // the item's records, requested before the stencil loads
    float4 Pn = stgP[0];
    for (int i = 0; i < n; ++i) {
        const float4 P = Pn;
        Pn = stgP[(i + 1) * NT];        // next record's first half (slot LMAX is readable: start of the float slots)
        CellWeights<O> w;
        w.set(P.x, P.y, P.z);
        float* o = stgF + i * NSLOT * NT;
        if constexpr ((MASK & 1) != 0) o[0 * NT] = st.template eval<0>(w);
        if constexpr ((MASK & 2) != 0) o[1 * NT] = st.template eval<1>(w);
        if constexpr ((MASK & 4) != 0) o[2 * NT] = st.template eval<2>(w);
        if constexpr ((MASK & 8) != 0) o[3 * NT] = st.template eval<3>(w);
        if constexpr ((MASK & 16) != 0) o[4 * NT] = st.template eval<4>(w);
        if constexpr ((MASK & 32) != 0) o[5 * NT] = st.template eval<5>(w);
    }
    __syncwarp();       // lanes with shorter items wait here: the next phase starts converged
}


// Work-item order for a supercell sorted in the prologue: cells by decreasing item length (a counting sort
// over min(length, 63); equal lengths in arrival order), first item of each.  perm/kbase as pic_sort_kernel
// publishes them, but in shared memory.
template <int NT>
__device__ __forceinline__ void fused_item_order(int tid, int seg_T, const int* s_off, int* s_w, int* s_bin /*[192]*/,
                                                 int* s_kcnt /*[256]*/, unsigned char* s_perm, unsigned short* s_kb)
{
    constexpr int PER = 256 / NT;
    int* s_base = s_bin + 64;
    int* s_bcur = s_bin + 128;
    for (int t = tid; t < 192; t += NT) s_bin[t] = 0;
    __syncthreads();
    int key[PER], kk[PER];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int c = tid * PER + k;
        const int n = s_off[c + 1] - s_off[c];
        kk[k] = (n + seg_T - 1) / seg_T;
        const int seglen = kk[k] ? (n + kk[k] - 1) / kk[k] : 0;
        key[k] = min(seglen, 63);
        atomicAdd(&s_bin[key[k]], 1);
    }
    __syncthreads();
    if (tid < 64) {
        int b = 0;
        for (int q = tid + 1; q < 64; ++q) b += s_bin[q];
        s_base[tid] = b;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int pos = s_base[key[k]] + atomicAdd(&s_bcur[key[k]], 1);
        s_perm[pos] = (unsigned char)(tid * PER + k);
        s_kcnt[pos] = kk[k];
    }
    __syncthreads();
    int v[PER], total;
#pragma unroll
    for (int k = 0; k < PER; ++k) v[k] = s_kcnt[tid * PER + k];
    block_excl_scan256<NT>(v, total, s_w, tid);
#pragma unroll
    for (int k = 0; k < PER; ++k) s_kb[tid * PER + k] = (unsigned short)min(v[k], 65535);
    __syncthreads();
}


}  // namespace
