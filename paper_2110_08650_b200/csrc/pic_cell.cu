// pic_cell.cu — the dense step kernel, third generation: one CTA of 128 threads per supercell,
// ONE THREAD OWNS ONE CELL for the step.  A warp takes 32 cells at a time, fullest cells first (so the 32 lanes
// walk similar numbers of particles); a thread walks its cell in near-equal chunks of at most LMAX particles:
//   phase 1 (a1-a3, a5)  the cell's stencil of three field components at a time sits in REGISTERS (TSC: Ex, By, Bz
//                        = 48 + 36 + 36 values, then Ey, Ez, Bx), contracted with each particle's weights as packed
//                        FMAs; the second pass adds the Boris push, the move and the in-place write-back (one
//                        32-byte store per record);
//   phase 2 (a4)         Esirkepov into 3 x 48 REGISTER sums over the cell's fixed 4x4x4-node window;
//   flush                the sums go into the shared split-integer J tile straight from the registers, every node at
//                        a compile-time offset from the window origin (two native ATOMS.ADD and ~4 other
//                        instructions per value, against ~13 through the staging column of the second generation).
// Against the second generation (pic_step.cu, MODE 2) there is no work-item list, crowded supercells need no
// separate one-phase variant, and the TSC weights are evaluated without floor / float->int conversions.
// Definitions: SURVEY.md §8(c) steps 1-7 (PAPER.md:60-62 names none of them).
#include <cuda.h>
#include <string.h>

#include "pic_step_common.cuh"

namespace {

#define PIC_CELL_THREADS 128
#define PIC_CELL_TBL 64          // frame-table entries kept in shared memory (16 k particles); beyond: global

// Shared memory of one supercell "stage": everything a CTA needs to step one supercell except the per-thread
// staging columns.  pic_cell_kernel has one stage; the persistent kernel two (the producer warps prepare the next
// supercell in one while the consumer warps step the current one in the other).
template <int O> struct CellStage {
    using G = Geo<O>;
    static constexpr int F_BYTES = 6 * G::FCOMP * 4;             // E/B tile [6][FNZ][FNY][FPX] (TMA destination)
    static constexpr int J_BYTES = 6 * G::JCOMP * 4;            // fixed-point pair (hi, lo)
    static constexpr int OFF_J = F_BYTES;
    static constexpr int OFF_CELLOFF = OFF_J + J_BYTES;          // int[260]
    static constexpr int OFF_HIST = OFF_CELLOFF + 260 * 4;       // int[256]
    static constexpr int OFF_ORDER = OFF_HIST + 256 * 4;         // u8[256] cells by decreasing population
    static constexpr int OFF_TBL = OFF_ORDER + 256;              // int[PIC_CELL_TBL]
    static constexpr int OFF_XREC = (OFF_TBL + PIC_CELL_TBL * 4 + 15) / 16 * 16;   // float4[2*XSTAGE]
    static constexpr int OFF_XID = OFF_XREC + PIC_XSTAGE * 32;   // u32[XSTAGE]
    static constexpr int OFF_XDST = OFF_XID + PIC_XSTAGE * 4;    // int[XSTAGE]
    static constexpr int OFF_SLOW = OFF_XDST + PIC_XSTAGE * 4;   // float[SLOWCAP][8]
    static constexpr int SLOWCAP = PIC_SLOWCAP_OF(O);
    static constexpr int OFF_VARS = OFF_SLOW + SLOWCAP * 32;     // int[16]: counters of the stage (CellVar)
    static constexpr int OFF_BARS = OFF_VARS + 64;               // u64[4]: mbarriers (tile, full, done)
    static constexpr int BYTES = (OFF_BARS + 32 + 127) / 128 * 128;
    // per thread and chunk slot the record's first half {fx,fy,fz,w} and NSLOT floats (gathered components on
    // their way to the Boris push, then the new position on its way to the deposit)
    static constexpr int LMAX = (O == 3) ? 7 : 12;
    static constexpr int NSLOT = (O == 3) ? 5 : 3;
    static_assert(LMAX + LMAX * NSLOT / 4 >= 12, "staging column too short for one component's sums");
    template <int NT> static constexpr int staging_bytes() { return LMAX * (16 + NSLOT * 4) * NT; }
};
enum CellVar { CV_XN = 0, CV_SLOWN, CV_XBASE, CV_NEXT, CV_NITEMS, CV_SC, CV_FIN, CV_COUNT };

// which components a gather pass holds in registers: the last pass is followed by the push
template <int O> struct CellPasses;
template <> struct CellPasses<1> { static constexpr int N = 1; static constexpr int M[6] = {0x3f, 0, 0, 0, 0, 0}; };
// TSC: Ex, By, Bz share the staggered x weights (48 + 36 + 36 registers), then Ey, Ez, Bx (48 + 48 + 36)
template <> struct CellPasses<2> { static constexpr int N = 2; static constexpr int M[6] = {0x31, 0x0e, 0, 0, 0, 0}; };
template <> struct CellPasses<3> { static constexpr int N = 6; static constexpr int M[6] = {0x01, 0x02, 0x04, 0x08, 0x10, 0x20}; };

template <int O> __host__ __device__ constexpr int cell_staged_mask() { return 0x3f & ~CellPasses<O>::M[CellPasses<O>::N - 1]; }
// staging slot of a component gathered before the last pass
template <int O> __host__ __device__ constexpr int cell_slot_of(int C)
{
    int n = 0;
    for (int c = 0; c < C; ++c) n += (cell_staged_mask<O>() >> c) & 1;
    return n;
}

// One gather pass over the n particles of the thread's chunk: the components in MASK, each into its staging slot.
template <int O, int MASK, int NSLOT, bool WAIT, int NT>
__device__ __forceinline__ void cell_gather_pass(const float* sF, int cx, int cy, int cz, int n, const float4* stgP, float* stgF)
{
    StencilSet<O, MASK> st;
    st.load(sF, cx, cy, cz);
    if (WAIT) cp_async_wait_all();      // the chunk's records, requested before the stencil loads
    float4 Pn = stgP[0];
    for (int i = 0; i < n; ++i) {
        const float4 P = Pn;
        Pn = stgP[(i + 1) * NT];        // next record's first half (slot LMAX is readable: start of the float slots)
        CellWeights<O> w;
        w.set(P.x, P.y, P.z);
        float* o = stgF + i * NSLOT * NT;
        if constexpr ((MASK & 1) != 0) o[cell_slot_of<O>(0) * NT] = st.template eval<0>(w);
        if constexpr ((MASK & 2) != 0) o[cell_slot_of<O>(1) * NT] = st.template eval<1>(w);
        if constexpr ((MASK & 4) != 0) o[cell_slot_of<O>(2) * NT] = st.template eval<2>(w);
        if constexpr ((MASK & 8) != 0) o[cell_slot_of<O>(3) * NT] = st.template eval<3>(w);
        if constexpr ((MASK & 16) != 0) o[cell_slot_of<O>(4) * NT] = st.template eval<4>(w);
        if constexpr ((MASK & 32) != 0) o[cell_slot_of<O>(5) * NT] = st.template eval<5>(w);
    }
    __syncwarp();       // lanes with shorter chunks wait here: the next phase starts converged
}

// Esirkepov weights of one particle over the cell's fixed 4-node window (nodes -1..2 per axis): S0 at the old
// in-cell position f0, DS = S1 - S0 with S1 at the new position x1 (relative to the old cell's origin node).
// Returns false when x1 leaves the window (the particle then takes the per-particle path).
template <int O>
__device__ __forceinline__ bool window_weights(const float (&f0)[3], const float (&x1)[3], float (&S0)[3][4], float (&DS)[3][4])
{
    bool fits = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float s1[4];
        if constexpr (O == 2) {
            fits &= (x1[a] >= -0.5f) & (x1[a] < 1.5f);
            tsc_window4(f0[a], S0[a]);
            tsc_window4(x1[a], s1);
        } else {
            float w0[O + 1], w1[O + 1];
            const int b0 = shape<O>(f0[a], w0);
            const int b1 = shape<O>(x1[a], w1);
            fits &= (b1 >= -1) & (b1 <= 2 - O);
            place4<O>(w0, b0 + 1, S0[a]);
            place4<O>(w1, b1 + 1, s1);
        }
#pragma unroll
        for (int t = 0; t < 4; ++t) DS[a][t] = s1[t] - S0[a][t];
    }
    return fits;
}

// register accumulation of one component over the cell's window, sums held as pairs over the b axis:
// A[i][b][c] += fac * (sum_{i'<=i} DS_a(i')) * (S0_b(b) C0_c(c) + DS_b(b) C1_c(c)),  i = nodes -1,0,1 of the flow axis,
// C0 = S0 + DS/2, C1 = S0/2 + DS/3 (the bracket, factored)
__device__ __forceinline__ void accumulate_pairs(f32x2 (&A)[3][2][4], float fac, const float (&DSa)[4],
                                                 const float (&S0b)[4], const float (&DSb)[4],
                                                 const float (&C0c)[4], const float (&C1c)[4])
{
    const float p0 = fac * DSa[0];
    const float p1 = fmaf(fac, DSa[1], p0);
    const float p2 = fmaf(fac, DSa[2], p1);
    const f32x2 P0 = pack2(p0, p0), P1 = pack2(p1, p1), P2 = pack2(p2, p2);
    const f32x2 s0[2] = {pack2(S0b[0], S0b[1]), pack2(S0b[2], S0b[3])};
    const f32x2 ds[2] = {pack2(DSb[0], DSb[1]), pack2(DSb[2], DSb[3])};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const f32x2 c0 = pack2(C0c[c], C0c[c]), c1 = pack2(C1c[c], C1c[c]);
#pragma unroll
        for (int bp = 0; bp < 2; ++bp) {
            const f32x2 br = fma2(s0[bp], c0, mul2(ds[bp], c1));
            A[0][bp][c] = fma2(P0, br, A[0][bp][c]);
            A[1][bp][c] = fma2(P1, br, A[1][bp][c]);
            A[2][bp][c] = fma2(P2, br, A[2][bp][c]);
        }
    }
}

// a5 for one particle, as finish_particle (pic_step_common.cuh) with the 32-byte store of store_record256
__device__ __forceinline__ void finish_particle256(const PicDev& d, float4* rec, size_t idx, int ssx, int ssy, int ssz,
                                                   int cx, int cy, int cz, int sp, float4 P, float4 M,
                                                   const float (&un)[3], const float (&fn)[3], const int (&sh)[3],
                                                   int* s_hist, int* s_xn, float4* s_xrec, uint32_t* s_xid, int* s_xdst)
{
    int ncx = cx + sh[0], ncy = cy + sh[1], ncz = cz + sh[2];
    const int dsx = (ncx < 0) ? -1 : (ncx >= PIC_SCX) ? 1 : 0;
    const int dsy = (ncy < 0) ? -1 : (ncy >= PIC_SCY) ? 1 : 0;
    const int dsz = (ncz < 0) ? -1 : (ncz >= PIC_SCZ) ? 1 : 0;
    ncx -= dsx * PIC_SCX; ncy -= dsy * PIC_SCY; ncz -= dsz * PIC_SCZ;
    const int nlc = ncx + PIC_SCX * (ncy + PIC_SCY * ncz);
    const uint32_t nbits = pic_pack_bits(nlc, sp);
    P.x = fn[0]; P.y = fn[1]; P.z = fn[2];
    M.x = un[0]; M.y = un[1]; M.z = un[2];
    M.w = __uint_as_float(nbits);
    if ((dsx | dsy | dsz) == 0) {
        store_record256(rec + 2 * idx, P, M);
        atomicAdd(&s_hist[nlc], 1);
    } else {
        const int dst = wrapi(ssx + dsx, d.nsx) + d.nsx * (wrapi(ssy + dsy, d.nsy) + d.nsy * wrapi(ssz + dsz, d.nsz));
        rec[2 * idx + 1] = make_float4(un[0], un[1], un[2], __uint_as_float(nbits | PIC_LEFT_FLAG));   // hole
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

// ------------------------------------------------------------------ one stage: views, prologue, batches, epilogue
template <int O> struct CellView {
    using G = Geo<O>;
    using S = CellStage<O>;
    float* sF; int* sJhi; int* sJlo; int* s_off; int* s_hist; unsigned char* s_order; int* s_tbl;
    float4* s_xrec; uint32_t* s_xid; int* s_xdst; float* s_slow; int* var; uint64_t* bars;
    __device__ __forceinline__ explicit CellView(unsigned char* b)
    {
        sF = reinterpret_cast<float*>(b);
        sJhi = reinterpret_cast<int*>(b + S::OFF_J);
        sJlo = sJhi + 3 * G::JCOMP;
        s_off = reinterpret_cast<int*>(b + S::OFF_CELLOFF);
        s_hist = reinterpret_cast<int*>(b + S::OFF_HIST);
        s_order = b + S::OFF_ORDER;
        s_tbl = reinterpret_cast<int*>(b + S::OFF_TBL);
        s_xrec = reinterpret_cast<float4*>(b + S::OFF_XREC);
        s_xid = reinterpret_cast<uint32_t*>(b + S::OFF_XID);
        s_xdst = reinterpret_cast<int*>(b + S::OFF_XDST);
        s_slow = reinterpret_cast<float*>(b + S::OFF_SLOW);
        var = reinterpret_cast<int*>(b + S::OFF_VARS);
        bars = reinterpret_cast<uint64_t*>(b + S::OFF_BARS);
    }
};

// try_wait with a suspend-time hint: a waiting warp sleeps in hardware instead of spinning through the issue slots
// the other role needs
__device__ __forceinline__ bool mbar_try_wait_hint(uint64_t* bar, unsigned parity, unsigned ns)
{
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(const PicDev& d, uint64_t* bar, unsigned parity)
{
    unsigned spins = 0;
    while (!mbar_try_wait_hint(bar, parity, 500u)) {
        if (++spins > (1u << 20)) {   // never hang the GPU on a lost arrival
            atomicOr(d.ctr + CTR_ERROR, PIC_DEV_TMA_TIMEOUT);
            break;
        }
    }
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Prepare supercell s in stage v (NT threads, barrier BAR): a2 stage the E/B tile, clear the J tile, a5 sort the
// previous step's result (or fetch the cell ranges of a sorted state), order the cells by population.
// bars[0] must be an initialised mbarrier (count 1) whose phase `tile_parity` is the one this load completes.
// Returns the supercell's population, or -1 after a sort mismatch (block-uniform).
template <int O, bool TMA, int NT, int BAR, int SORT_R>
__device__ __forceinline__ int cell_prologue(const PicDev& d, const CUtensorMap* tmap, const CellView<O>& v, int s, int tid,
                                             unsigned tile_parity)
{
    using G = Geo<O>;
    using S = CellStage<O>;
    const int ssx = s % d.nsx, ssy = (s / d.nsx) % d.nsy, ssz = s / (d.nsx * d.nsy);
    const int ox = ssx * PIC_SCX, oy = ssy * PIC_SCY, oz = ssz * PIC_SCZ;
    if (TMA) {
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the tile's last readers were generic loads
            mbar_expect_tx(v.bars, 6u * G::FCOMP * sizeof(float));
            tma_load_4d(v.sF, tmap, v.bars, ox /* pad_lo_x == FL: 16 B aligned */, oy + PIC_PAD_LO - G::FL,
                        oz + PIC_PAD_LO - G::FL, 0);
        }
    } else {
        for (int e = tid; e < 6 * G::FNZ * G::FNY * G::FNX; e += NT) {
            int i = e % G::FNX;
            int r = e / G::FNX;
            int j = r % G::FNY;
            r /= G::FNY;
            int k = r % G::FNZ;
            int c = r / G::FNZ;
            int gi = wrapi(ox + i - G::FL, d.nx), gj = wrapi(oy + j - G::FL, d.ny),
                gk = wrapi(oz + k - G::FL, d.nz);
            v.sF[c * G::FCOMP + (k * G::FNY + j) * G::FPX + i] =
                __ldg(d.Fpad + pic_padded_index(d, c, gi, gj, gk));
        }
    }
    // scratch of the fused sort and of the cell order: the leaver staging area, unused until the particle loop
    int* s_w = reinterpret_cast<int*>(v.s_xrec);                           // [16]
    int* s_bin = s_w + 16;                                                 // [192]
    static_assert((16 + PIC_SORT_TBL) * 4 <= PIC_XSTAGE * 40, "frame table scratch must fit the leaver staging area");
    if (d.fused) {
        // SORT_R > 0: records staged through the J tile area (free until the tile is cleared below)
        static_assert(SORT_R * NT * 36 <= S::J_BYTES, "sort staging must fit the J tile");
        if (fused_sort<NT, BAR, 4, SORT_R>(d, s, tid, v.s_off, v.s_hist, s_w, s_w + 16, reinterpret_cast<unsigned char*>(v.sJhi)) < 0)
            return -1;     // block-uniform
        group_sync<BAR, NT>();
    } else {
        for (int t = tid; t < 257; t += NT) v.s_off[t] = d.cell_off[(size_t)s * 257 + t];
    }
    for (int e = tid; e < 6 * G::JCOMP; e += NT) v.sJhi[e] = 0;
    for (int t = tid; t < 256; t += NT) v.s_hist[t] = 0;
    for (int t = tid; t < 192; t += NT) s_bin[t] = 0;
    if (tid == 0) {
        v.var[CV_XN] = 0;
        v.var[CV_SLOWN] = 0;
        v.var[CV_NEXT] = 0;
        v.var[CV_FIN] = 0;
    }
    group_sync<BAR, NT>();
    const int count = v.s_off[256];
    {
        const int nfr = min((count + PIC_FRAME - 1) / PIC_FRAME, PIC_CELL_TBL);
        for (int t = tid; t < nfr; t += NT) v.s_tbl[t] = d.tbl_pool[d.tbl_off[s] + t];
    }
    // cells by decreasing population (a counting sort over min(population, 63); equal populations in arrival
    // order): the 32 cells a warp takes at a time hold similar numbers of particles
    {
        int* s_base = s_bin + 64;
        int* s_bcur = s_bin + 128;
        int key[256 / NT];
#pragma unroll
        for (int k = 0; k < 256 / NT; ++k) {
            const int c = tid * (256 / NT) + k;
            key[k] = min(v.s_off[c + 1] - v.s_off[c], 63);
            atomicAdd(&s_bin[key[k]], 1);
        }
        group_sync<BAR, NT>();
        if (tid < 64) {
            int b = 0;
            for (int q = tid + 1; q < 64; ++q) b += s_bin[q];
            s_base[tid] = b;
        }
        if (tid == 0) {
            v.var[CV_NITEMS] = 256 - s_bin[0];       // empty cells come last and are not taken
            v.var[CV_COUNT] = count;
        }
        group_sync<BAR, NT>();
#pragma unroll
        for (int k = 0; k < 256 / NT; ++k) {
            const int pos = s_base[key[k]] + atomicAdd(&s_bcur[key[k]], 1);
            v.s_order[pos] = (unsigned char)(tid * (256 / NT) + k);
        }
    }
    group_sync<BAR, NT>();
    if (TMA) mbar_wait(d, v.bars, tile_parity);
    return count;
}

// The particle work of one supercell for one warp: it takes 32 cells at a time until none is left.
// stgP / stgF: this thread's staging column (stride NT between a column's slots).
template <int O, int NT>
__device__ __forceinline__ void cell_batches(const PicDev& d, const CellView<O>& v, int s, float4* const stgP, float* const stgF,
                                             int lane, const float (&jfs)[3])
{
    using G = Geo<O>;
    using S = CellStage<O>;
    const int ssx = s % d.nsx, ssy = (s / d.nsx) % d.nsy, ssz = s / (d.nsx * d.nsy);
    float4* rec = d.rec[d.cur];
    const float* sF = v.sF;
    const int* gtbl = d.tbl_pool + d.tbl_off[s];
    auto record_index = [&](int slot) -> size_t {
        const int fr = slot >> 8;
        const int f = (fr < PIC_CELL_TBL) ? v.s_tbl[fr] : gtbl[fr];
        return (size_t)f * PIC_FRAME + (slot & (PIC_FRAME - 1));
    };
    const int n_items = v.var[CV_NITEMS];
    constexpr int SX = 1, SY = G::JNX, SZ = G::JNX * G::JNY;

    for (;;) {   // a warp takes 32 cells at a time
        int ibase = 0;
        if (lane == 0) ibase = atomicAdd(&v.var[CV_NEXT], 32);
        ibase = __shfl_sync(0xffffffffu, ibase, 0);
        if (ibase >= n_items) break;
        const bool has = ibase + lane < n_items;
        const int lc = has ? v.s_order[ibase + lane] : 0;
        const int p0 = v.s_off[lc];
        const int n_tot = has ? v.s_off[lc + 1] - p0 : 0;
        const int cx = lc & 7, cy = (lc >> 3) & 7, cz = lc >> 6;
        // near-equal chunks of at most LMAX particles
        const int n_chunks = (n_tot + S::LMAX - 1) / S::LMAX;
        const int q_len = n_chunks ? n_tot / n_chunks : 0, r_len = n_chunks ? n_tot % n_chunks : 0;

        int done = 0;
        for (int ch = 0; __any_sync(0xffffffffu, ch < n_chunks); ++ch) {
            const int n = (ch < n_chunks) ? q_len + (ch < r_len) : 0;
            const int p = p0 + done;
            // ---- phase 1, a1: request the records' first halves into the thread's own column
            for (int i = 0; i < n; ++i) cp_async16(stgP + i * NT, rec + 2 * record_index(p + i));
            // ---- a2: gather passes with the stencil in registers; the last one adds a3 + a5
            using CP = CellPasses<O>;
            if constexpr (CP::N >= 2) cell_gather_pass<O, CP::M[0], S::NSLOT, true, NT>(sF, cx, cy, cz, n, stgP, stgF);
            if constexpr (CP::N >= 3) cell_gather_pass<O, CP::M[1], S::NSLOT, false, NT>(sF, cx, cy, cz, n, stgP, stgF);
            if constexpr (CP::N >= 4) cell_gather_pass<O, CP::M[2], S::NSLOT, false, NT>(sF, cx, cy, cz, n, stgP, stgF);
            if constexpr (CP::N >= 5) cell_gather_pass<O, CP::M[3], S::NSLOT, false, NT>(sF, cx, cy, cz, n, stgP, stgF);
            if constexpr (CP::N >= 6) cell_gather_pass<O, CP::M[4], S::NSLOT, false, NT>(sF, cx, cy, cz, n, stgP, stgF);
            {
                constexpr int LAST = CP::M[CP::N - 1];
                StencilSet<O, LAST> st;
                st.load(sF, cx, cy, cz);
                if constexpr (CP::N == 1) cp_async_wait_all();
                size_t idx_n = 0;
                float4 Mn = make_float4(0.f, 0.f, 0.f, 0.f);
                if (n > 0) {
                    idx_n = record_index(p);
                    Mn = rec[2 * idx_n + 1];
                }
                float4 Pn = stgP[0];
                for (int i = 0; i < n; ++i) {
                    const size_t idx = idx_n;
                    const float4 M = Mn;
                    if (i + 1 < n) {
                        idx_n = record_index(p + i + 1);
                        Mn = rec[2 * idx_n + 1];
                    }
                    const float4 P = Pn;
                    Pn = stgP[(i + 1) * NT];
                    float* o = stgF + i * S::NSLOT * NT;
                    CellWeights<O> w;
                    w.set(P.x, P.y, P.z);
                    float E[3], B[3];
                    if constexpr ((LAST & 1) != 0) E[0] = st.template eval<0>(w); else E[0] = o[cell_slot_of<O>(0) * NT];
                    if constexpr ((LAST & 2) != 0) E[1] = st.template eval<1>(w); else E[1] = o[cell_slot_of<O>(1) * NT];
                    if constexpr ((LAST & 4) != 0) E[2] = st.template eval<2>(w); else E[2] = o[cell_slot_of<O>(2) * NT];
                    if constexpr ((LAST & 8) != 0) B[0] = st.template eval<3>(w); else B[0] = o[cell_slot_of<O>(3) * NT];
                    if constexpr ((LAST & 16) != 0) B[1] = st.template eval<4>(w); else B[1] = o[cell_slot_of<O>(4) * NT];
                    if constexpr ((LAST & 32) != 0) B[2] = st.template eval<5>(w); else B[2] = o[cell_slot_of<O>(5) * NT];
                    const int sp = (__float_as_uint(M.w) >> 16) & 0xff;
                    float un[3], fn[3], x1[3];
                    int sh[3];
                    boris_move(d, sp, P, M, E, B, un, fn, x1, sh);
                    o[0 * NT] = x1[0]; o[1 * NT] = x1[1]; o[2 * NT] = x1[2];
                    reinterpret_cast<float*>(stgP + i * NT)[3] = d.q[sp] * P.w;
                    finish_particle256(d, rec, idx, ssx, ssy, ssz, cx, cy, cz, sp, P, M, un, fn, sh, v.s_hist, &v.var[CV_XN],
                                       v.s_xrec, v.s_xid, v.s_xdst);
                }
                __syncwarp();
            }
            // ---- phase 2, a4: Esirkepov into the register sums.  (They cannot outlive the chunk: 144 sums plus the
            // 120-132 stencil registers of phase 1 do not fit the 255 registers of a thread.)
            f32x2 Ax[3][2][4], Ay[3][2][4], Az[3][2][4];     // sums over (flow node, pair of b nodes, c node)
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int b = 0; b < 2; ++b)
#pragma unroll
                    for (int c = 0; c < 4; ++c) Ax[i][b][c] = Ay[i][b][c] = Az[i][b][c] = 0ull;
            {
                float4 Pn = stgP[0];     // {f0, q*w}
                float xn[3] = {stgF[0 * NT], stgF[1 * NT], stgF[2 * NT]};
                for (int i = 0; i < n; ++i) {
                    const float4 P = Pn;
                    const float f0[3] = {P.x, P.y, P.z};
                    const float x1[3] = {xn[0], xn[1], xn[2]};
                    Pn = stgP[(i + 1) * NT];
                    if (i + 1 < S::LMAX) {              // (keeps the prefetch inside the float slots)
                        const float* o = stgF + (i + 1) * S::NSLOT * NT;
                        xn[0] = o[0 * NT]; xn[1] = o[1 * NT]; xn[2] = o[2 * NT];
                    }
                    const float qw = P.w;
                    float S0[3][4], DS[3][4];
                    if (window_weights<O>(f0, x1, S0, DS)) {
                        float C0[3][4], C1[3][4];
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int t = 0; t < 4; ++t) {
                                C0[a][t] = S0[a][t] + 0.5f * DS[a][t];
                                C1[a][t] = 0.5f * S0[a][t] + (1.0f / 3.0f) * DS[a][t];
                            }
                        accumulate_pairs(Ax, -qw * jfs[0], DS[0], S0[1], DS[1], C0[2], C1[2]);
                        accumulate_pairs(Ay, -qw * jfs[1], DS[1], S0[2], DS[2], C0[0], C1[0]);
                        accumulate_pairs(Az, -qw * jfs[2], DS[2], S0[0], DS[0], C0[1], C1[1]);
                    } else {
                        const int k = atomicAdd(&v.var[CV_SLOWN], 1);
                        if (k < S::SLOWCAP) {
                            float* q = v.s_slow + 8 * k;
                            q[0] = f0[0]; q[1] = f0[1]; q[2] = f0[2];
                            q[3] = x1[0]; q[4] = x1[1]; q[5] = x1[2];
                            q[6] = qw; q[7] = __int_as_float(lc);
                        } else {            // queue full: hand the particle to pic_overflow_kernel
                            const int k2 = atomicAdd(d.ctr + CTR_OVF, 1);
                            if (k2 < d.ovf_cap) {
                                d.ovf[2 * (size_t)k2] = make_float4(f0[0], f0[1], f0[2], qw);
                                d.ovf[2 * (size_t)k2 + 1] = make_float4(x1[0], x1[1], x1[2], __int_as_float(lc | (s << 8)));
                            } else {
                                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_OVERFLOW_QUEUE_FULL);
                            }
                        }
                    }
                }
                __syncwarp();
            }
            done += n;
            // ---- a4: one flush of the chunk's 3 x 48 sums into the shared fixed-point tile, through the thread's own
            // staging column and a rolled loop over the components (the unrolled form is 14 KB of code and was
            // measured slower: together with the phase loops it overflows the instruction cache).
            // Rows (i,b) of four values: the first LMAX rows in the float4 slots, the rest in the float slots.
            if (n > 0) {
                const int j0 = (cx - 1 + G::JL) * SX + (cy - 1 + G::JL) * SY + (cz - 1 + G::JL) * SZ;
#pragma unroll 1
                for (int comp = 0; comp < 3; ++comp) {
                    auto stage_sums = [&](const f32x2 (&A)[3][2][4]) {
#pragma unroll
                        for (int r = 0; r < 12; ++r) {
                            const int i = r >> 2, b = r & 3;
                            float q[4];
#pragma unroll
                            for (int c = 0; c < 4; ++c) {
                                float lo, hi;
                                unpack2(A[i][b >> 1][c], lo, hi);
                                q[c] = (b & 1) ? hi : lo;
                            }
                            if (r < S::LMAX) stgP[r * NT] = make_float4(q[0], q[1], q[2], q[3]);
                            else {
#pragma unroll
                                for (int c = 0; c < 4; ++c) stgF[((r - S::LMAX) * 4 + c) * NT] = q[c];
                            }
                        }
                    };
                    if (comp == 0) stage_sums(Ax);
                    else if (comp == 1) stage_sums(Ay);
                    else stage_sums(Az);
                    const int sa = comp == 0 ? SX : comp == 1 ? SY : SZ;
                    const int sb = comp == 0 ? SY : comp == 1 ? SZ : SX;
                    const int sc = comp == 0 ? SZ : comp == 1 ? SX : SY;
                    const int cbase = j0 + comp * G::JCOMP;
                    constexpr int RP = S::LMAX < 12 ? S::LMAX : 12;     // rows kept in the float4 slots
                    float4 qn = stgP[0];
#pragma unroll 1
                    for (int r = 0; r < RP; ++r) {
                        const float4 q = qn;
                        qn = stgP[(r + 1) * NT];
                        const int rb = cbase + (r >> 2) * sa + (r & 3) * sb;
                        fix_add2(v.sJhi, v.sJlo, rb, rb + sc, q.x, q.y);
                        fix_add2(v.sJhi, v.sJlo, rb + 2 * sc, rb + 3 * sc, q.z, q.w);
                    }
#pragma unroll 1
                    for (int r = RP; r < 12; ++r) {
                        const float* f = stgF + (r - RP) * 4 * NT;
                        const int rb = cbase + (r >> 2) * sa + (r & 3) * sb;
                        fix_add2(v.sJhi, v.sJlo, rb, rb + sc, f[0], f[NT]);
                        fix_add2(v.sJhi, v.sJlo, rb + 2 * sc, rb + 3 * sc, f[2 * NT], f[3 * NT]);
                    }
                }
            }
            __syncwarp();
        }
    }   // next batch of cells
}

// a4: the stage's queued out-of-window particles, one thread each (NT threads whose warps all take part)
template <int O, int NT>
__device__ __forceinline__ void cell_slow_queue(const PicDev& d, const CellView<O>& v, int tid, const float (&fix_scale)[3])
{
    using S = CellStage<O>;
    const int n_slow = min(v.var[CV_SLOWN], S::SLOWCAP);
    for (int base = 0; base < n_slow; base += NT) {
        if (base + (tid & ~31) < n_slow) {          // warp-uniform
            const int e = base + tid;
            float f0[3] = {0.5f, 0.5f, 0.5f}, x1[3] = {0.5f, 0.5f, 0.5f}, qw = 0.0f;
            int qlc = 0;
            if (e < n_slow) {
                const float* q = v.s_slow + 8 * e;
                f0[0] = q[0]; f0[1] = q[1]; f0[2] = q[2];
                x1[0] = q[3]; x1[1] = q[4]; x1[2] = q[5];
                qw = q[6]; qlc = __float_as_int(q[7]);
            }
            deposit_direct<O, true>(d, reinterpret_cast<float*>(v.sJhi), v.sJhi, v.sJlo, fix_scale, f0, x1, qw, qlc);
        }
    }
}

// a5 + a4 at the end of a supercell (NT threads, barrier BAR): leavers staged in shared memory -> one append to the
// exchange buffer; stayers per new cell; the J tile -> global 64-bit fixed-point accumulators (native RED.64).
template <int O, int NT, int BAR>
__device__ __forceinline__ void cell_epilogue(const PicDev& d, const CellView<O>& v, int s, int tid)
{
    using G = Geo<O>;
    const int ssx = s % d.nsx, ssy = (s / d.nsx) % d.nsy, ssz = s / (d.nsx * d.nsy);
    const int ox = ssx * PIC_SCX, oy = ssy * PIC_SCY, oz = ssz * PIC_SCZ;
    const int s_xn = v.var[CV_XN];
    const int n_x = min(s_xn, PIC_XSTAGE);
    if (tid == 0) d.sc_left[s] = s_xn;          // every leaver, staged or appended directly (pic_prepare_kernel)
    if (tid == 0 && n_x > 0) v.var[CV_XBASE] = atomicAdd(d.ctr + CTR_EXCH, n_x);
    group_sync<BAR, NT>();
    const int xbase = v.var[CV_XBASE];
    for (int k = tid; k < n_x; k += NT) {
        const int xs = xbase + k;
        if (xs < d.x_cap) {
            d.x_rec[2 * (size_t)xs] = v.s_xrec[2 * k];
            d.x_rec[2 * (size_t)xs + 1] = v.s_xrec[2 * k + 1];
            d.x_id[xs] = d.pid[d.cur][v.s_xid[k]];      // staged: the record index (< 2^32 slots)
            d.x_dst[xs] = v.s_xdst[k];
        } else {
            atomicOr(d.ctr + CTR_ERROR, PIC_DEV_EXCHANGE_OVERFLOW);
        }
    }
    // stayers per new cell (neighbours add their leavers to the same counters)
    for (int t = tid; t < 256; t += NT)
        if (v.s_hist[t] != 0) atomicAdd(d.cell_hist + (size_t)s * 256 + t, v.s_hist[t]);
    // the J tile (periodic wrap on write): 16 lanes per row of JNX <= 13 nodes
    const size_t ncell = (size_t)d.nx * d.ny * d.nz;
    constexpr int ROWS = 3 * G::JNZ * G::JNY;
    const int i = tid & 15;
    if (i < G::JNX) {
        const int gi = wrapi(ox + i - G::JL, d.nx);
        for (int row = tid >> 4; row < ROWS; row += NT / 16) {
            const int e = row * G::JNX + i;
            const long long n = ((long long)v.sJhi[e] << PIC_FIX_LO_BITS) + (long long)v.sJlo[e];
            if (n == 0) continue;
            const int j = row % G::JNY;
            const int r2 = row / G::JNY;
            const int k = r2 % G::JNZ;
            const int c = r2 / G::JNZ;
            const int gj = wrapi(oy + j - G::JL, d.ny), gk = wrapi(oz + k - G::JL, d.nz);
            const size_t g = c * ncell + (size_t)gi + (size_t)d.nx * ((size_t)gj + (size_t)d.ny * gk);
            atomicAdd(reinterpret_cast<unsigned long long*>(d.J64) + g, (unsigned long long)n);
        }
    }
}

__device__ __forceinline__ bool cell_is_dense(const PicDev& d, int s);
// next dense supercell from the global work counter, or -1
__device__ __forceinline__ int fetch_work(const PicDev& d)
{
    int s;
    do {
        s = atomicAdd(d.ctr + CTR_WORK, 1);
    } while (s < d.nsc && !cell_is_dense(d, s));
    return s < d.nsc ? s : -1;
}
__device__ __forceinline__ bool cell_is_dense(const PicDev& d, int s)
{
    // the supercell's population: after the pending sort (fused prologue), or as sorted
    const int n = d.fused ? d.sc_next[s] : d.sc_count[s];
    if (n == 0) {
        retire_empty_supercell(d, s);      // (called by one thread per supercell: thread 0 of its CTA, or the fetching thread)
        return false;
    }
    const bool sparse_class = d.class_all == 1 || (d.class_all == 0 && n < d.direct_below);
    return !sparse_class;
}

// ------------------------------------------------------------------ kernel 1: one CTA of 128 threads per supercell
template <int O, bool TMA>
__global__ void __launch_bounds__(PIC_CELL_THREADS, 2)
pic_cell_kernel(const PicDev d, const __grid_constant__ CUtensorMap tmap)
{
    constexpr int NT = PIC_CELL_THREADS;
    using S = CellStage<O>;
    const int s = pic_cta_supercell(d, blockIdx.x);
    if (s < 0) return;
    {
        __shared__ int s_dense;
        if (threadIdx.x == 0) s_dense = cell_is_dense(d, s);
        __syncthreads();
        if (!s_dense) return;
    }
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const CellView<O> v(smem_raw);
    float4* s_stgP = reinterpret_cast<float4*>(smem_raw + S::BYTES);
    float* s_stgF = reinterpret_cast<float*>(smem_raw + S::BYTES + S::LMAX * 16 * NT);
    const int tid = threadIdx.x;
    if (TMA && tid == 0) mbar_init(v.bars, 1);
    __syncthreads();
    if (cell_prologue<O, TMA, NT, 0, 0>(d, &tmap, v, s, tid, 0) < 0) return;

    float fix_scale[3];
    fix_scale[0] = fix_scale_of(d, d.jfx);
    fix_scale[1] = fix_scale_of(d, d.jfy);
    fix_scale[2] = fix_scale_of(d, d.jfz);
    const float jfs[3] = {d.jfx * fix_scale[0], d.jfy * fix_scale[1], d.jfz * fix_scale[2]};
    cell_batches<O, NT>(d, v, s, s_stgP + tid, s_stgF + tid, tid & 31, jfs);
    __syncthreads();
    cell_slow_queue<O, NT>(d, v, tid, fix_scale);
    __syncthreads();
    cell_epilogue<O, NT, 0>(d, v, s, tid);
}

// ------------------------------------------------------------------ kernel 2: persistent, warp-specialized
// One CTA per SM, three warp groups.  The PRODUCER group (128 threads, registers cut to PIC_PRODUCER_REGS) fetches
// supercells from a global counter and, for each, prepares one of two stages: TMA tile, J tile clear, the counting
// sort of the previous step's result, the cell order; and it retires finished stages: leaver append, histogram,
// J tile flush.  The two CONSUMER groups (256 threads, registers raised to PIC_CONSUMER_REGS) run cell_batches on
// the ready stage and move on to the next one without a CTA-wide barrier: the HBM- and latency-bound sort and the
// tile flush run beside the FP-bound particle work instead of in front of and behind it.
//   full[b]  producer -> consumers  stage b is prepared (its supercell index in var[CV_SC]; -1 = no more work)
//   done[b]  consumers -> producer  every consumer warp has left stage b (and its slow queue is deposited)
#define PIC_P_THREADS 384
#define PIC_P_CONSUMERS 256
#define PIC_PRODUCER_REGS 56
#define PIC_CONSUMER_REGS 224
enum { BAR_TILE = 0, BAR_FULL = 1, BAR_DONE = 2 };

template <int O, bool TMA>
__global__ void __launch_bounds__(PIC_P_THREADS, 1)
pic_pcell_kernel(const PicDev d, const __grid_constant__ CUtensorMap tmap)
{
    using S = CellStage<O>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const CellView<O> v0(smem_raw), v1(smem_raw + S::BYTES);
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int b = 0; b < 2; ++b) {
            uint64_t* bars = b ? v1.bars : v0.bars;
            mbar_init(bars + BAR_TILE, 1);
            mbar_init(bars + BAR_FULL, 1);
            mbar_init(bars + BAR_DONE, 1);
        }
    }
    __syncthreads();

    if (tid >= PIC_P_CONSUMERS) {
        // ============================================================ producer group
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PIC_PRODUCER_REGS));
        constexpr int NT = PIC_P_THREADS - PIC_P_CONSUMERS;
        const int ptid = tid - PIC_P_CONSUMERS;
        __shared__ int s_work[2];
        int live[2] = {-1, -1};           // stage b: >= 0 supercell to retire, -3 handed over but skipped, -1 free
        unsigned use[2] = {0, 0};         // how often stage b has been prepared and handed to the consumers
        bool more = true;
        for (int k = 0;; ++k) {
            const int b = k & 1;
            const CellView<O>& v = b ? v1 : v0;
            // retire the supercell that used this stage two rounds ago
            if (live[b] != -1) {
                mbar_wait(d, v.bars + BAR_DONE, (use[b] - 1) & 1);
                if (live[b] >= 0) cell_epilogue<O, NT, 1>(d, v, live[b], ptid);
                group_sync<1, NT>();
                live[b] = -1;
            }
            if (!more) {
                if (live[b ^ 1] == -1) break;
                continue;
            }
            // next dense supercell, fetched one ahead: the one after it is prefetched into L2 while this one is sorted
            // (the sort's record loads are what the producer waits for)
            if (ptid == 0) {
                if (k == 0) s_work[1] = fetch_work(d);
                s_work[0] = s_work[1];
                s_work[1] = s_work[0] >= 0 ? fetch_work(d) : -1;
            }
            group_sync<1, NT>();
            const int s = s_work[0], s_ahead = s_work[1];
            group_sync<1, NT>();
            if (s_ahead >= 0 && d.fused) {
                const int n_scan = d.sc_tail[s_ahead];
                const int* tb = d.tbl_pool + d.tbl_off[s_ahead];
                const float4* src = d.rec[d.cur ^ 1];
                const uint32_t* sid = d.pid[d.cur ^ 1];
                for (int l = ptid; l < (n_scan + 3) / 4; l += NT) {          // one 128-byte line = 4 records
                    const int slot = 4 * l;
                    const size_t i = (size_t)tb[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(src + 2 * i));
                    if ((l & 7) == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(sid + i));      // 32 ids per line
                }
            }
            if (s < 0) {                  // no more work: the consumers leave when they reach this stage
                more = false;
                if (ptid == 0) {
                    v.var[CV_SC] = -1;
                    mbar_arrive(v.bars + BAR_FULL);
                }
                continue;
            }
            const int rc = cell_prologue<O, TMA, NT, 1, (S::J_BYTES / (NT * 36) < 7 ? S::J_BYTES / (NT * 36) : 7)>(d, &tmap, v, s, ptid, use[b] & 1);
            if (ptid == 0) {
                v.var[CV_SC] = rc < 0 ? -2 : s;        // -2: sort mismatch (the sticky error is set): nothing to step
                mbar_arrive(v.bars + BAR_FULL);
            }
            live[b] = rc < 0 ? -3 : s;
            ++use[b];
        }
    } else {
        // ============================================================ consumer groups
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(PIC_CONSUMER_REGS));
        constexpr int NT = PIC_P_CONSUMERS;
        float4* s_stgP = reinterpret_cast<float4*>(smem_raw + 2 * S::BYTES);
        float* s_stgF = reinterpret_cast<float*>(smem_raw + 2 * S::BYTES + S::LMAX * 16 * NT);
        const int lane = tid & 31;
        float fix_scale[3];
        fix_scale[0] = fix_scale_of(d, d.jfx);
        fix_scale[1] = fix_scale_of(d, d.jfy);
        fix_scale[2] = fix_scale_of(d, d.jfz);
        const float jfs[3] = {d.jfx * fix_scale[0], d.jfy * fix_scale[1], d.jfz * fix_scale[2]};
        unsigned use[2] = {0, 0};
        for (int k = 0;; ++k) {
            const int b = k & 1;
            const CellView<O>& v = b ? v1 : v0;
            mbar_wait(d, v.bars + BAR_FULL, use[b] & 1);
            ++use[b];
            const int s = v.var[CV_SC];
            if (s == -1) break;
            if (s >= 0) cell_batches<O, NT>(d, v, s, s_stgP + tid, s_stgF + tid, lane, jfs);
            // the last warp to leave the stage deposits its queued out-of-window particles and hands it back
            __syncwarp();
            int fin = 0;
            if (lane == 0) {
                __threadfence_block();
                fin = atomicAdd(&v.var[CV_FIN], 1);
            }
            fin = __shfl_sync(0xffffffffu, fin, 0);
            if (fin == PIC_P_CONSUMERS / 32 - 1) {
                __threadfence_block();
                if (s >= 0) cell_slow_queue<O, 32>(d, v, lane, fix_scale);
                __syncwarp();
                if (lane == 0) {
                    v.var[CV_FIN] = 0;
                    __threadfence_block();
                    mbar_arrive(v.bars + BAR_DONE);
                }
            }
        }
    }
}

}  // namespace

template <int O, bool TMA>
static cudaError_t launch_cell_one(const PicDev& d, const CUtensorMap& map, cudaStream_t st)
{
    static bool configured = false;     // opt in to > 48 KB of dynamic shared memory once
    constexpr int bytes = CellStage<O>::BYTES + CellStage<O>::template staging_bytes<PIC_CELL_THREADS>();
    static_assert(2 * (bytes + 1024 + 256) <= 228 * 1024, "two cell CTAs must fit one SM");
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(pic_cell_kernel<O, TMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        int ctas = 0;                   // the design point is two CTAs per SM
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, pic_cell_kernel<O, TMA>, PIC_CELL_THREADS, bytes);
        if (e != cudaSuccess) return e;
        if (ctas < 2) return cudaErrorLaunchOutOfResources;
        configured = true;
    }
    pic_cell_kernel<O, TMA><<<pic_step_grid(d), PIC_CELL_THREADS, bytes, st>>>(d, map);
    return cudaGetLastError();
}

template <int O, bool TMA>
static cudaError_t launch_pcell_one(const PicDev& d, const CUtensorMap& map, cudaStream_t st)
{
    static int n_sm = 0;
    constexpr int bytes = 2 * CellStage<O>::BYTES + CellStage<O>::template staging_bytes<PIC_P_CONSUMERS>();
    static_assert(bytes <= 227 * 1024, "the persistent CTA must fit one SM");
    if (n_sm == 0) {
        cudaError_t e = cudaFuncSetAttribute(pic_pcell_kernel<O, TMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        int dev = 0, ctas = 0;
        e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, pic_pcell_kernel<O, TMA>, PIC_P_THREADS, bytes);
        if (e != cudaSuccess) { n_sm = 0; return e; }
        if (ctas < 1) { n_sm = 0; return cudaErrorLaunchOutOfResources; }
    }
    pic_pcell_kernel<O, TMA><<<n_sm < d.nsc ? n_sm : d.nsc, PIC_P_THREADS, bytes, st>>>(d, map);
    return cudaGetLastError();
}

cudaError_t pic_launch_cell(const PicDev& d, int order, bool use_tma, const void* tmap, cudaStream_t st, int64_t* launches,
                            bool persistent)
{
    CUtensorMap map;
    if (use_tma) memcpy(&map, tmap, sizeof map); else memset(&map, 0, sizeof map);
    cudaError_t e;
#define PIC_GO(O)                                                                                                    \
    e = persistent ? (use_tma ? launch_pcell_one<O, true>(d, map, st) : launch_pcell_one<O, false>(d, map, st))       \
                   : (use_tma ? launch_cell_one<O, true>(d, map, st) : launch_cell_one<O, false>(d, map, st))
    switch (order) {
        case 1: PIC_GO(1); break;
        case 2: PIC_GO(2); break;
        default: PIC_GO(3); break;
    }
#undef PIC_GO
    ++*launches;
    return e;
}
