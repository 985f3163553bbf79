// pic_step.cu — the step kernels of the first two generations and the kernels around the step.
// pic_step_kernel<O, TMA, FIX, MODE>, one CTA per supercell, particles sorted by cell:
//   MODE 1 (sparse, 256 threads): one thread per particle, Esirkepov straight into the shared tile — the variant
//          every step still launches for supercells with fewer than 6 particles per cell;
//   MODE 2 (two-phase, 128 threads): work items of <= LMAX particles, cell stencils and Esirkepov sums in registers;
//   MODE 0 (one-phase, 128 threads): gather per particle from the shared tile, register sums per cell segment.
// MODE 0 and 2 are the dense kernels of round 1, kept as selectable variants (option "cell_kernel" = 0); the default
// dense kernel is pic_cell_kernel (pic_cell.cu).  Also here: overflow queue, J conversion, frame bookkeeping
// (prepare), leaver scatter, the stand-alone counting sort.
// Definitions: SURVEY.md §8(c) steps 1-7 (PAPER.md:60-62 names none of them).
#include <cuda.h>
#include <string.h>

#include "pic_step_common.cuh"

namespace {


template <int O, bool FIX> struct StepSmem {
    using G = Geo<O>;
    static constexpr int F_BYTES = 6 * G::FCOMP * 4;
    static constexpr int J_BYTES = (FIX ? 6 : 3) * G::JCOMP * 4;
    static constexpr int OFF_J = F_BYTES;
    static constexpr int OFF_CELLOFF = OFF_J + J_BYTES;          // int[260]
    static constexpr int OFF_HIST = OFF_CELLOFF + 260 * 4;       // int[256]
    static constexpr int OFF_XREC = (OFF_HIST + 256 * 4 + 15) / 16 * 16;   // float4[2*XSTAGE]
    static constexpr int OFF_XID = OFF_XREC + PIC_XSTAGE * 32;   // u32[XSTAGE]
    static constexpr int OFF_XDST = OFF_XID + PIC_XSTAGE * 4;    // int[XSTAGE]
    static constexpr int OFF_SLOW = OFF_XDST + PIC_XSTAGE * 4;   // float[SLOWCAP][8]
    static constexpr int SLOWCAP = PIC_SLOWCAP_OF(O);
    static constexpr int OFF_ITEMS = OFF_SLOW + SLOWCAP * 32;    // int2[ITEMCAP]
    // two-phase path: per thread and item slot the record's first half {fx,fy,fz,w} and NSLOT floats
    // (gathered components on their way to the Boris push, then the new position on its way to the deposit)
    static constexpr int LMAX = PIC_ITEM_LMAX(O);
    static constexpr int NSLOT = (O == 3) ? 5 : 3;
    static constexpr int OFF_STGP = (OFF_ITEMS + PIC_ITEMCAP * 8 + 15) / 16 * 16;   // float4[LMAX][128]
    static constexpr int OFF_STGF = OFF_STGP + LMAX * 16 * PIC_STEP_THREADS;         // float[LMAX][NSLOT][128]
    static constexpr int TOTAL = OFF_STGF + LMAX * NSLOT * 4 * PIC_STEP_THREADS;
    // two CTAs per SM: 228 KB of shared memory, 1 KB reserved per CTA, < 256 B of static variables
    // (checked again at run time by launch_step_one: the kernel must reach 2 CTAs per SM)
    static_assert(!FIX || 2 * (TOTAL + 1024 + 256) <= 228 * 1024, "two step CTAs must fit one SM");
};


// ------------------------------------------------------------------ the step kernel
// MODE 2: supercells with >= PIC_DIRECT_BELOW particles whose work items fit the two-phase path (<= LMAX
//         particles each): 128 threads, per-cell stencils and Esirkepov sums in registers.
// MODE 0: more crowded supercells (or two_phase off): 128 threads, gather per particle from the shared
//         tile, register sums per cell segment.
// MODE 1: sparse supercells, 256 threads, one thread per particle straight into the tile.
// Every variant is launched over all supercells; a CTA whose supercell belongs to another one exits.
#define PIC_MODE_ONE 0
#define PIC_MODE_SPARSE 1
#define PIC_MODE_TWO 2
template <int O, bool TMA, bool FIX, int MODE>
__global__ void __launch_bounds__(MODE == PIC_MODE_SPARSE ? 256 : PIC_STEP_THREADS, MODE == PIC_MODE_SPARSE ? 3 : 2)
pic_step_kernel(const PicDev d, const __grid_constant__ CUtensorMap tmap)
{
    constexpr bool SPARSE = MODE == PIC_MODE_SPARSE;
    constexpr bool two_phase = MODE == PIC_MODE_TWO;
    constexpr int NT = SPARSE ? 256 : PIC_STEP_THREADS;
    const int s = pic_cta_supercell(d, blockIdx.x);
    if (s < 0) return;
    {
        // the supercell's population: after the pending sort (fused prologue), or as sorted
        const int n = d.fused ? d.sc_next[s] : d.sc_count[s];
        if (n == 0) {
            if (threadIdx.x == 0) retire_empty_supercell(d, s);
            return;
        }
        const bool sparse_class = d.class_all == 1 || (d.class_all == 0 && n < d.direct_below);
        if (sparse_class != SPARSE) return;
        if (!SPARSE) {
            const bool fits_two = d.two_phase && pic_segment_target(n, d.seg_num, PIC_ITEM_LMAX(O)) <= PIC_ITEM_LMAX(O);
            if (fits_two != two_phase) return;
        }
    }
    using G = Geo<O>;
    using S = StepSmem<O, FIX>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sF = reinterpret_cast<float*>(smem_raw);                 // E/B tile [6][FNZ][FNY][FPX]
    float* sJ = reinterpret_cast<float*>(smem_raw + S::OFF_J);      // float J tile [3][JNZ][JNY][JNX]
    int* sJhi = reinterpret_cast<int*>(sJ);                         // or the fixed-point pair
    int* sJlo = sJhi + 3 * G::JCOMP;
    int* s_off = reinterpret_cast<int*>(smem_raw + S::OFF_CELLOFF);
    int* s_hist = reinterpret_cast<int*>(smem_raw + S::OFF_HIST);
    float4* s_xrec = reinterpret_cast<float4*>(smem_raw + S::OFF_XREC);
    uint32_t* s_xid = reinterpret_cast<uint32_t*>(smem_raw + S::OFF_XID);
    int* s_xdst = reinterpret_cast<int*>(smem_raw + S::OFF_XDST);
    float* s_slow = reinterpret_cast<float*>(smem_raw + S::OFF_SLOW);
    int2* s_items = reinterpret_cast<int2*>(smem_raw + S::OFF_ITEMS);
    float4* s_stgP = reinterpret_cast<float4*>(smem_raw + S::OFF_STGP);
    float* s_stgF = reinterpret_cast<float*>(smem_raw + S::OFF_STGF);
    __shared__ int s_xn, s_slown, s_xbase, s_next, s_nitems;
    __shared__ int s_any;        // sparse variant: some particle of the supercell deposited
    __shared__ int s_tbl[two_phase ? (768 * PIC_ITEM_LMAX(O)) / PIC_FRAME + 3 : 1];
    __shared__ __align__(8) uint64_t s_bar;

    const int tid = threadIdx.x;
    const int ssx = s % d.nsx, ssy = (s / d.nsx) % d.nsy, ssz = s / (d.nsx * d.nsy);
    const int ox = ssx * PIC_SCX, oy = ssy * PIC_SCY, oz = ssz * PIC_SCZ;
    constexpr int NJ = (FIX ? 6 : 3) * G::JCOMP;
    float4* rec = d.rec[d.cur];

    // ---- a2: stage the E/B tile, clear the J tile, fetch the cell ranges
    if (TMA) {
        if (tid == 0) {
            mbar_init(&s_bar, 1);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&s_bar, 6u * G::FCOMP * sizeof(float));
            tma_load_4d(sF, &tmap, &s_bar, ox /* pad_lo_x == FL: 16 B aligned */, oy + PIC_PAD_LO - G::FL,
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
            sF[c * G::FCOMP + (k * G::FNY + j) * G::FPX + i] =
                __ldg(d.Fpad + pic_padded_index(d, c, gi, gj, gk));
        }
    }
    for (int e = tid; e < NJ; e += NT) sJhi[e] = 0;
    // scratch of the fused sort: the leaver staging area, unused until the particle loop
    int* s_w = reinterpret_cast<int*>(smem_raw + S::OFF_XREC);             // [16]
    int* s_bin = s_w + 16;                                                 // [192]
    int* s_kcnt = s_bin + 192;                                             // [256]
    unsigned char* s_perm = reinterpret_cast<unsigned char*>(s_kcnt + 256);       // [256]
    unsigned short* s_kb = reinterpret_cast<unsigned short*>(s_perm + 256);       // [256]
    static_assert((16 + 192 + 256) * 4 + 256 + 512 <= PIC_XSTAGE * 40, "sort scratch must fit the leaver staging area");
    static_assert((16 + PIC_SORT_TBL) * 4 <= PIC_XSTAGE * 40, "frame table scratch must fit the leaver staging area");
    // sparse supercells (3 CTAs of 256 threads per SM: too few warps to hide the sort's latencies) were
    // sorted by pic_sort_kernel just before this launch
    const bool fused = !SPARSE && d.fused != 0;
    if (fused) {
        if (fused_sort<NT>(d, s, tid, s_off, s_hist, s_w, s_w + 16) < 0) return;     // block-uniform
        __syncthreads();
    } else {
        for (int t = tid; t < 257; t += NT) s_off[t] = d.cell_off[(size_t)s * 257 + t];
    }
    for (int t = tid; t < 256; t += NT) s_hist[t] = 0;
    if (tid == 0) {
        s_xn = 0;
        s_slown = 0;
        s_next = 0;
        s_any = 0;
    }
    __syncthreads();
    // work items: every cell is cut into k = ceil(n/T) near-equal segments, T ~ 3/4 of the mean cell
    // population; cells come in the order the sort kernel fixed (by decreasing segment length), so
    // the 32 items a warp takes at a time hold similar numbers of particles
    const int seg_T = pic_segment_target(s_off[256], d.seg_num, d.two_phase ? PIC_ITEM_LMAX(O) : 0);
    if constexpr (two_phase) {
        const int nfr = (s_off[256] + PIC_FRAME - 1) / PIC_FRAME;
        if (tid < nfr) s_tbl[tid] = d.tbl_pool[d.tbl_off[s] + tid];
    }
    // the item order: published by pic_sort_kernel for the supercells it counts as dense, else worked out here
    // (after the fused sort; or a supercell below the line that this variant takes under class_all == 2)
    const bool own_order = fused || s_off[256] < d.direct_below;
    if (!SPARSE && own_order) fused_item_order<NT>(tid, seg_T, s_off, s_w, s_bin, s_kcnt, s_perm, s_kb);
    if (!SPARSE)
    for (int t = tid; t < 256; t += NT) {
        const int c = own_order ? s_perm[t] : d.cell_perm[(size_t)s * 256 + t];
        const int n = s_off[c + 1] - s_off[c];
        const int k = (n + seg_T - 1) / seg_T;
        int at = own_order ? s_kb[t] : d.cell_kbase[(size_t)s * 256 + t];
        if (t == 255) s_nitems = min(at + k, PIC_ITEMCAP);
        const int q = k ? n / k : 0, r = k ? n % k : 0;
        int start = s_off[c];
        for (int j = 0; j < k && at < PIC_ITEMCAP; ++j, ++at) {
            const int len = q + (j < r);
            s_items[at] = make_int2(start, (len << 8) | c);
            start += len;
        }
    }
    __syncthreads();
    if (TMA) {
        unsigned spins = 0;
        while (!mbar_try_wait(&s_bar, 0)) {
            if (++spins > (1u << 20)) {   // never hang the GPU on a lost copy
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_TMA_TIMEOUT);
                break;
            }
        }
    }

    // Sparse variant: is the staged E/B tile all zero (plasma the fields have not reached)?  A particle at rest
    // (u = 0 exactly) in such a supercell gathers F = 0, keeps u = 0 and x, and deposits nothing: the step leaves its
    // record bit for bit as it is, so only the cell histogram has to hear of it (see the particle loop).
    bool tile_zero = false;
    if (SPARSE && d.rest_skip) {
        unsigned any = 0;
        for (int e = tid; e < 6 * G::FCOMP; e += NT) any |= __float_as_uint(sF[e]) << 1;     // -0 counts as zero
        tile_zero = __syncthreads_or(any != 0) == 0;
    }

    float fix_scale[3] = {1.0f, 1.0f, 1.0f};
    if (FIX) {
        fix_scale[0] = fix_scale_of(d, d.jfx);
        fix_scale[1] = fix_scale_of(d, d.jfy);
        fix_scale[2] = fix_scale_of(d, d.jfz);
    }
    const float jfs[3] = {d.jfx * fix_scale[0], d.jfy * fix_scale[1], d.jfz * fix_scale[2]};

    // frame table: the two-phase variant (<= 768*LMAX particles, i.e. <= 35 frames) reads it from shared memory
    const int* tbl = d.tbl_pool + d.tbl_off[s];
    if constexpr (two_phase) tbl = s_tbl;
    const int lane = tid & 31;
    const int n_items = s_nitems;
    constexpr int SX = 1, SY = G::JNX, SZ = G::JNX * G::JNY;

    // (no-sort step, sparse variant only: the slots in use — stayers, holes of earlier leavers, appended arrivals —
    // are walked as they are; the variant needs no cell order)
    const int count = (SPARSE && d.nosort) ? min(d.sc_tail[s], d.sc_nframes[s] * PIC_FRAME) : s_off[256];
    if (SPARSE) {
        // sparse supercell (a few particles per cell): register sums would be flushed almost once per
        // particle, so take one thread per particle, coalesced, and deposit straight into the tile.
        // (Tried: the first batch's records — population -> frame table -> record, three dependent loads — requested
        // at the top of the prologue, beside the tile copy: configs[2] 5.97 instead of 5.82 ms per step.)
        for (int base = 0; base < count; base += NT) {
            if (base + (tid & ~31) >= count) continue;       // warp-uniform
            const int slot = base + tid;
            bool active = slot < count;
            float4 P = make_float4(0.5f, 0.5f, 0.5f, 0.0f), M = make_float4(0.f, 0.f, 0.f, 0.f);   // ghost lane
            size_t idx = 0;
            if (active) {
                idx = (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
                load_record256(rec + 2 * idx, P, M);
                if (__float_as_uint(M.w) & PIC_LEFT_FLAG) {      // hole of a particle that left in an earlier step
                    active = false;
                    P = make_float4(0.5f, 0.5f, 0.5f, 0.0f);
                    M = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
            const uint32_t bits = __float_as_uint(M.w);
            const int lc = bits & 0xff, sp = (bits >> 16) & 0xff;
            const int cx = lc & 7, cy = (lc >> 3) & 7, cz = lc >> 6;
            // a warp of particles at rest in a field-free supercell: nothing to compute, nothing to write back
            const bool at_rest = tile_zero && ((__float_as_uint(M.x) | __float_as_uint(M.y) | __float_as_uint(M.z)) << 1) == 0;
            if (__all_sync(0xffffffffu, at_rest || !active)) {
                if (active) atomicAdd(&s_hist[lc], 1);
                continue;
            }
            float un[3], fn[3], x1[3];
            int sh[3];
            push_particle<O>(d, sF, cx, cy, cz, sp, P, M, un, fn, x1, sh);
            const float f0[3] = {P.x, P.y, P.z};
            // a particle whose position did not change in fp32 deposits exactly nothing (every DS is 0): a warp of
            // such particles (cold plasma ahead of a laser pulse) skips the deposit altogether
            const bool moved = (x1[0] != f0[0]) | (x1[1] != f0[1]) | (x1[2] != f0[2]);
            if (__any_sync(0xffffffffu, moved)) {
                if (lane == 0) s_any = 1;
                deposit_direct<O, FIX>(d, sJ, sJhi, sJlo, fix_scale, f0, x1, d.q[sp] * P.w, lc);
            }
            if (active)
                finish_particle(d, rec, idx, s, ssx, ssy, ssz, cx, cy, cz, sp, P, M, un, fn, sh, s_hist, &s_xn, s_xrec,
                                s_xid, s_xdst);
        }
    } else
    for (;;) {   // a warp takes 32 work items at a time
    int ibase = 0;
    if (lane == 0) ibase = atomicAdd(&s_next, 32);
    ibase = __shfl_sync(0xffffffffu, ibase, 0);
    if (ibase >= n_items) break;
    int p = 0, p_end = 0, lc = 0;
    if (ibase + lane < n_items) {
        const int2 it = s_items[ibase + lane];
        p = it.x;
        p_end = it.x + (it.y >> 8);
        lc = it.y & 0xff;
    }
    const int cx = lc & 7, cy = (lc >> 3) & 7, cz = lc >> 6;
    float Ax[3][4][4], Ay[3][4][4], Az[3][4][4];

    // a4 for one particle of the item: Esirkepov, accumulated in registers over the cell's window
    // (nodes -1..2); a particle whose new position leaves the window is queued
    auto deposit_in_window = [&](const float (&f0)[3], const float (&x1)[3], float qw) {
        float S0[3][4], DS[3][4];
        bool fits = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float s1[4];
            if constexpr (O == 2) {         // TSC: the window weights without floor / float->int / index compares
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
        if (fits) {
            accumulate1(Ax, -qw * jfs[0], DS[0], S0[1], DS[1], S0[2], DS[2]);
            accumulate1(Ay, -qw * jfs[1], DS[1], S0[2], DS[2], S0[0], DS[0]);
            accumulate1(Az, -qw * jfs[2], DS[2], S0[0], DS[0], S0[1], DS[1]);
        } else {
            const int k = atomicAdd(&s_slown, 1);
            if (k < S::SLOWCAP) {
                float* q = s_slow + 8 * k;
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
    };
    auto zero_sums = [&]() {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int c = 0; c < 4; ++c) Ax[i][b][c] = Ay[i][b][c] = Az[i][b][c] = 0.0f;
    };

    if constexpr (two_phase) {
        // ---- two-phase item (<= LMAX particles).  Phase 1, a2 + a3 + a5: the cell's stencil of a few
        // components at a time sits in REGISTERS while the thread walks its particles; gathered values
        // wait in the thread's own shared-memory column.  Phase 2, a4: the register sums.  The two
        // phases never hold their registers (stencils / sums) at the same time.
        constexpr int LAST = (O == 1) ? 0x3f : (O == 2) ? 0x38 : 0x20;    // components gathered in the last pass
        const int n = p_end - p;
        float4* stgP = s_stgP + tid;
        float* stgF = s_stgF + tid;
        for (int i = 0; i < n; ++i) {
            const size_t idx = (size_t)tbl[(p + i) >> 8] * PIC_FRAME + ((p + i) & (PIC_FRAME - 1));
            cp_async16(stgP + i * NT, rec + 2 * idx);
        }
        if constexpr (O == 2) gather_pass<O, 0x07, S::NSLOT, true>(sF, cx, cy, cz, n, stgP, stgF);
        if constexpr (O == 3) {
            gather_pass<O, 0x01, S::NSLOT, true>(sF, cx, cy, cz, n, stgP, stgF);
            gather_pass<O, 0x02, S::NSLOT, false>(sF, cx, cy, cz, n, stgP, stgF);
            gather_pass<O, 0x04, S::NSLOT, false>(sF, cx, cy, cz, n, stgP, stgF);
            gather_pass<O, 0x08, S::NSLOT, false>(sF, cx, cy, cz, n, stgP, stgF);
            gather_pass<O, 0x10, S::NSLOT, false>(sF, cx, cy, cz, n, stgP, stgF);
        }
        {
            StencilSet<O, LAST> st;
            st.load(sF, cx, cy, cz);
            if constexpr (O == 1) cp_async_wait_all();
            size_t idx_n = 0;
            float4 Mn = make_float4(0.f, 0.f, 0.f, 0.f);
            if (n > 0) {
                idx_n = (size_t)tbl[p >> 8] * PIC_FRAME + (p & (PIC_FRAME - 1));
                Mn = rec[2 * idx_n + 1];
            }
            float4 Pn = stgP[0];
            for (int i = 0; i < n; ++i) {
                const size_t idx = idx_n;
                const float4 M = Mn;
                if (i + 1 < n) {
                    idx_n = (size_t)tbl[(p + i + 1) >> 8] * PIC_FRAME + ((p + i + 1) & (PIC_FRAME - 1));
                    Mn = rec[2 * idx_n + 1];
                }
                const float4 P = Pn;
                Pn = stgP[(i + 1) * NT];
                float* o = stgF + i * S::NSLOT * NT;
                CellWeights<O> w;
                w.set(P.x, P.y, P.z);
                float E[3], B[3];
                if constexpr ((LAST & 1) != 0) E[0] = st.template eval<0>(w); else E[0] = o[0 * NT];
                if constexpr ((LAST & 2) != 0) E[1] = st.template eval<1>(w); else E[1] = o[1 * NT];
                if constexpr ((LAST & 4) != 0) E[2] = st.template eval<2>(w); else E[2] = o[2 * NT];
                if constexpr ((LAST & 8) != 0) B[0] = st.template eval<3>(w); else B[0] = o[3 * NT];
                if constexpr ((LAST & 16) != 0) B[1] = st.template eval<4>(w); else B[1] = o[4 * NT];
                B[2] = st.template eval<5>(w);
                const int sp = (__float_as_uint(M.w) >> 16) & 0xff;
                float un[3], fn[3], x1[3];
                int sh[3];
                boris_move(d, sp, P, M, E, B, un, fn, x1, sh);
                o[0 * NT] = x1[0]; o[1 * NT] = x1[1]; o[2 * NT] = x1[2];
                reinterpret_cast<float*>(stgP + i * NT)[3] = d.q[sp] * P.w;
                finish_particle(d, rec, idx, s, ssx, ssy, ssz, cx, cy, cz, sp, P, M, un, fn, sh, s_hist, &s_xn, s_xrec,
                                s_xid, s_xdst);
            }
            __syncwarp();
        }
        zero_sums();
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
            deposit_in_window(f0, x1, P.w);
        }
        __syncwarp();
    } else {
    zero_sums();
    // the next record is fetched while the current particle is processed
    size_t idx_n = 0;
    float4 Pn = make_float4(0.f, 0.f, 0.f, 0.f), Mn = Pn;
    if (p < p_end) {
        idx_n = (size_t)tbl[p >> 8] * PIC_FRAME + (p & (PIC_FRAME - 1));
        Pn = rec[2 * idx_n];
        Mn = rec[2 * idx_n + 1];
    }
    for (; p < p_end; ++p) {
        const size_t idx = idx_n;
        float4 P = Pn, M = Mn;
        if (p + 1 < p_end) {
            idx_n = (size_t)tbl[(p + 1) >> 8] * PIC_FRAME + ((p + 1) & (PIC_FRAME - 1));
            Pn = rec[2 * idx_n];
            Mn = rec[2 * idx_n + 1];
        }
        const int sp = (__float_as_uint(M.w) >> 16) & 0xff;
        float un[3], fn[3], x1[3];
        int sh[3];
        push_particle<O>(d, sF, cx, cy, cz, sp, P, M, un, fn, x1, sh);
        const float f0[3] = {P.x, P.y, P.z};
        deposit_in_window(f0, x1, d.q[sp] * P.w);
        finish_particle(d, rec, idx, s, ssx, ssy, ssz, cx, cy, cz, sp, P, M, un, fn, sh, s_hist, &s_xn, s_xrec, s_xid, s_xdst);
    }
    }

    // ---- a4: one flush of the item's 3 x 48 partial sums into the shared tile
    if (ibase + lane < n_items) {
        const int j0 = (cx - 1 + G::JL) * SX + (cy - 1 + G::JL) * SY + (cz - 1 + G::JL) * SZ;
        if constexpr (two_phase) {
            // through the thread's own staging column and a rolled loop: the unrolled form is 18 KB of
            // code, which together with the three phase loops overflows the 32 KB instruction cache
            // rows (i,b) of four values: the first LMAX rows in the float4 slots, the rest in the float slots
            static_assert(S::LMAX + S::LMAX * S::NSLOT / 4 >= 12, "staging column too short for one component's sums");
            float4* colP = s_stgP + tid;
            float* colF = s_stgF + tid;
#pragma unroll 1
            for (int comp = 0; comp < 3; ++comp) {
                auto stage_sums = [&](const float (&A)[3][4][4]) {
#pragma unroll
                    for (int r = 0; r < 12; ++r) {
                        const int i = r >> 2, b = r & 3;
                        if (r < S::LMAX) colP[r * NT] = make_float4(A[i][b][0], A[i][b][1], A[i][b][2], A[i][b][3]);
                        else {
#pragma unroll
                            for (int c = 0; c < 4; ++c) colF[((r - S::LMAX) * 4 + c) * NT] = A[i][b][c];
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
                float4 qn = colP[0];
#pragma unroll 1
                for (int r = 0; r < RP; ++r) {
                    const float4 q = qn;
                    qn = colP[(r + 1) * NT];
                    const int rb = cbase + (r >> 2) * sa + (r & 3) * sb;
                    flush2<FIX>(sJ, sJhi, sJlo, rb, rb + sc, q.x, q.y);
                    flush2<FIX>(sJ, sJhi, sJlo, rb + 2 * sc, rb + 3 * sc, q.z, q.w);
                }
#pragma unroll 1
                for (int r = RP; r < 12; ++r) {
                    const float* f = colF + (r - RP) * 4 * NT;
                    const int rb = cbase + (r >> 2) * sa + (r & 3) * sb;
                    flush2<FIX>(sJ, sJhi, sJlo, rb, rb + sc, f[0], f[NT]);
                    flush2<FIX>(sJ, sJhi, sJlo, rb + 2 * sc, rb + 3 * sc, f[2 * NT], f[3 * NT]);
                }
            }
        } else {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    flush1<FIX>(sJ, sJhi, sJlo, j0 + 0 * G::JCOMP + i * SX + b * SY + c * SZ, Ax[i][b][c]);
                    flush1<FIX>(sJ, sJhi, sJlo, j0 + 1 * G::JCOMP + i * SY + b * SZ + c * SX, Ay[i][b][c]);
                    flush1<FIX>(sJ, sJhi, sJlo, j0 + 2 * G::JCOMP + i * SZ + b * SX + c * SY, Az[i][b][c]);
                }
        }
    }
    }   // next batch of work items
    __syncthreads();

    // ---- a4: queued out-of-window particles, one thread each
    {
        const int n_slow = min(s_slown, S::SLOWCAP);
        for (int base = 0; base < n_slow; base += NT) {
            if (base + (tid & ~31) < n_slow) {          // warp-uniform
                const int e = base + tid;
                float f0[3] = {0.5f, 0.5f, 0.5f}, x1[3] = {0.5f, 0.5f, 0.5f}, qw = 0.0f;
                int qlc = 0;
                if (e < n_slow) {
                    const float* q = s_slow + 8 * e;
                    f0[0] = q[0]; f0[1] = q[1]; f0[2] = q[2];
                    x1[0] = q[3]; x1[1] = q[4]; x1[2] = q[5];
                    qw = q[6]; qlc = __float_as_int(q[7]);
                }
                deposit_direct<O, FIX>(d, sJ, sJhi, sJlo, fix_scale, f0, x1, qw, qlc);
            }
        }
    }

    // ---- a5: leavers staged in shared memory -> one append to the exchange buffer
    const int n_x = min(s_xn, PIC_XSTAGE);
    if (tid == 0) d.sc_left[s] = s_xn;          // every leaver, staged or appended directly (pic_prepare_kernel)
    if (tid == 0 && n_x > 0) s_xbase = atomicAdd(d.ctr + CTR_EXCH, n_x);
    __syncthreads();
    for (int k = tid; k < n_x; k += NT) {
        const int xs = s_xbase + k;
        if (xs < d.x_cap) {
            d.x_rec[2 * (size_t)xs] = s_xrec[2 * k];
            d.x_rec[2 * (size_t)xs + 1] = s_xrec[2 * k + 1];
            d.x_id[xs] = d.pid[d.cur][s_xid[k]];      // staged: the record index (< 2^32 slots)
            d.x_dst[xs] = s_xdst[k];
        } else {
            atomicOr(d.ctr + CTR_ERROR, PIC_DEV_EXCHANGE_OVERFLOW);
        }
    }
    // stayers per new cell (neighbours add their leavers to the same counters)
    for (int t = tid; t < 256; t += NT)
        if (s_hist[t] != 0) atomicAdd(d.cell_hist + (size_t)s * 256 + t, s_hist[t]);

    // ---- a4: flush the J tile once (periodic wrap on write)
    // A sparse supercell none of whose particles moved (cold plasma ahead of a laser pulse) has an all-zero tile: no
    // flush.  And a node is read before its address is worked out: at 1.5 particles per cell most nodes of a tile are
    // zero, and the walk over the 3456 nodes was 38 % of the sparse variant's instructions on configs[2] (ncu).
    if (!SPARSE || s_any) {
        // A row of the tile (component, z, y) maps to a row of the global array: its cell offset — two divisions, two
        // periodic wraps, three multiplications — is worked out once per row into a table (in the leaver staging area,
        // free by now), not once per node: the per-node version spent 44 instructions behind every non-zero node
        // (ncu, hot-spot variant: 228 of 2044 thread instructions per particle).  32-bit offsets: pic_create admits at
        // most 2^22 supercells = 2^30 cells, and 3 x 2^30 < 2^32.
        constexpr int ROWS = 3 * G::JNZ * G::JNY;
        static_assert(ROWS * 4 <= PIC_XSTAGE * 40, "row table must fit the leaver staging area");
        unsigned* s_rowbase = reinterpret_cast<unsigned*>(smem_raw + S::OFF_XREC);
        const unsigned ncell = (unsigned)d.nx * (unsigned)d.ny * (unsigned)d.nz;
        __syncthreads();                 // the append above has read the staging area
        for (int row = tid; row < ROWS; row += NT) {
            const int j = row % G::JNY;
            const int r2 = row / G::JNY;
            const int k = r2 % G::JNZ;
            const int c = r2 / G::JNZ;
            const int gj = wrapi(oy + j - G::JL, d.ny), gk = wrapi(oz + k - G::JL, d.nz);
            s_rowbase[row] = (unsigned)c * ncell + (unsigned)d.nx * ((unsigned)gj + (unsigned)d.ny * (unsigned)gk);
        }
        __syncthreads();
        // 16 lanes per tile row of JNX <= 13 nodes
        const int i = tid & 15;
        const unsigned gi = (unsigned)wrapi(ox + i - G::JL, d.nx);
        if (i < G::JNX)
        for (int row = tid >> 4; row < ROWS; row += NT / 16) {
            const int e = row * G::JNX + i;
            long long n = 0;
            float v = 0.0f;
            if (FIX) {
                n = ((long long)sJhi[e] << PIC_FIX_LO_BITS) + (long long)sJlo[e];
                if (n == 0) continue;
            } else {
                v = sJ[e];
                if (v == 0.0f) continue;
            }
            const size_t g = (size_t)(s_rowbase[row] + gi);
            if (FIX) {
                // 64-bit fixed point in global memory too (native RED.64 in L2)
                atomicAdd(reinterpret_cast<unsigned long long*>(d.J64) + g, (unsigned long long)n);
            } else if (d.float_tile_to_j64) {
                // float tile of a sparse supercell (few same-node collisions: the CAS loop of a float atomic is
                // cheaper there than two integer atomics) into the fixed-point global accumulators
                const int c = row / (G::JNY * G::JNZ);
                const float jfc = c == 0 ? d.jfx : c == 1 ? d.jfy : d.jfz;
                const double scale = (double)fix_scale_of(d, jfc) * (double)(1 << PIC_FIX_LO_BITS);
                atomicAdd(reinterpret_cast<unsigned long long*>(d.J64) + g, (unsigned long long)__double2ll_rn((double)v * scale));
            } else {
                atomicAdd(d.J + g, v);
            }
        }
    }
}

// Out-of-window particles that did not fit a CTA's shared-memory queue: one thread per particle,
// Esirkepov straight into the global accumulators (rare: needs > 768 such particles in one supercell).
template <int O, bool FIX>
__global__ void pic_overflow_kernel(const PicDev d)
{
    const int n = min(d.ctr[CTR_OVF], d.ovf_cap);
    const size_t ncell = (size_t)d.nx * d.ny * d.nz;
    const float jf[3] = {d.jfx, d.jfy, d.jfz};
    const int dims[3] = {d.nx, d.ny, d.nz};
    const size_t stride[3] = {1, (size_t)d.nx, (size_t)d.nx * d.ny};
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const float4 A = d.ovf[2 * (size_t)e], Bq = d.ovf[2 * (size_t)e + 1];
        const float f0[3] = {A.x, A.y, A.z}, x1[3] = {Bq.x, Bq.y, Bq.z};
        const float qw = A.w;
        const int code = __float_as_int(Bq.w);
        const int lc = code & 255, s = code >> 8;
        const int cell[3] = {(s % d.nsx) * PIC_SCX + (lc & 7), ((s / d.nsx) % d.nsy) * PIC_SCY + ((lc >> 3) & 7),
                             (s / (d.nsx * d.nsy)) * PIC_SCZ + (lc >> 6)};
        float S0[3][O + 2], DS[3][O + 2];
        int lo[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float w0[O + 1], w1[O + 1], s1[O + 2];
            const int b0 = shape<O>(f0[a], w0), b1 = shape<O>(x1[a], w1);
            lo[a] = min(b0, b1);
            to_window<O>(w0, b0 - lo[a], S0[a]);
            to_window<O>(w1, b1 - lo[a], s1);
#pragma unroll
            for (int t = 0; t < O + 2; ++t) DS[a][t] = s1[t] - S0[a][t];
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int b = (a + 1) % 3, c = (a + 2) % 3;
            const float scale = FIX ? fix_scale_of(d, jf[a]) : 1.0f;
            const float fac = -qw * jf[a] * scale;
            for (int tc = 0; tc < O + 2; ++tc)
                for (int tb = 0; tb < O + 2; ++tb) {
                    const float br = fac * (S0[b][tb] * S0[c][tc] + 0.5f * DS[b][tb] * S0[c][tc] +
                                            0.5f * S0[b][tb] * DS[c][tc] + (1.0f / 3.0f) * DS[b][tb] * DS[c][tc]);
                    float acc = 0.0f;
                    for (int ta = 0; ta < O + 1; ++ta) {
                        acc = fmaf(DS[a][ta], br, acc);
                        if (acc == 0.0f) continue;
                        int idx[3];
                        idx[a] = cell[a] + lo[a] + ta; idx[b] = cell[b] + lo[b] + tb; idx[c] = cell[c] + lo[c] + tc;
                        size_t g = a * ncell;
#pragma unroll
                        for (int x = 0; x < 3; ++x) g += stride[x] * (size_t)wrapi(idx[x], dims[x]);
                        if (FIX)
                            atomicAdd(reinterpret_cast<unsigned long long*>(d.J64) + g,
                                      (unsigned long long)__double2ll_rn((double)acc * (double)(1 << PIC_FIX_LO_BITS)));
                        else
                            atomicAdd(d.J + g, acc);
                    }
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

// ------------------------------------------------------------------ resort
// One thread per supercell: make sure the frame list can hold the slots in use (holes of
// leavers stay until the sort) plus the arrivals appended behind them.
__global__ void pic_prepare_kernel(const PicDev d)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.nsc) return;
    // slots in use: the sorted population, or — after a step that ran without a sort — everything up to the tail
    // (holes stay until the next sort; arrivals are appended behind them)
    const int count = d.nosort ? d.sc_tail[s] : d.sc_count[s];
    const int inc = d.sc_incoming[s];
    const int need = (count + inc + PIC_FRAME - 1) / PIC_FRAME;
    int have = d.sc_nframes[s];
    if (need > have) {
        int off = d.tbl_off[s];
        if (need > d.tbl_cap[s]) {
            // Grow the frame table: capacities are powers of two, a region of the right class is taken from the free
            // lists if one is there (this kernel only pops — a CAS loop, no pushes run beside it — and
            // pic_reclaim_tables_kernel, launched right after this one, only pushes), else cut from the pool.  The old region goes
            // back to its class (a general allocator with reclaim).
            const int ocap = d.tbl_cap[s];
            int want = max(2 * ocap, need + 4), k = 3;
            while ((1 << k) < want) ++k;
            const int ncap = 1 << k;
            int noff = -1;
            for (int t = d.tbl_free_top[k]; t > 0;) {
                const int seen = atomicCAS(d.tbl_free_top + k, t, t - 1);
                if (seen == t) {
                    noff = d.tbl_free[k * PIC_TBL_FREE + t - 1];
                    break;
                }
                t = seen;
            }
            if (noff < 0) {
                noff = atomicAdd(d.ctr + CTR_TBL_TOP, ncap);
                if (noff + ncap > d.tbl_pool_size) {
                    atomicOr(d.ctr + CTR_ERROR, PIC_DEV_TABLE_POOL_EXHAUSTED);
                    return;
                }
            }
            for (int i = 0; i < have; ++i) d.tbl_pool[noff + i] = d.tbl_pool[off + i];
            if (ocap > 0) {
                d.tbl_old_off[s] = off;
                d.tbl_old_cap[s] = ocap;
            }
            d.tbl_off[s] = off = noff;
            d.tbl_cap[s] = ncap;
        }
        // returned frames first (this kernel only pops, the sort kernel only pushes; the counter may
        // dip below zero here and is clamped by the next kernel), then fresh ones from the pool
        for (int i = have; i < need; ++i) {
            int f;
            const int t = atomicSub(d.ctr + CTR_FREE_TOP, 1);
            if (t > 0) {
                f = d.free_stack[t - 1];
            } else {
                f = atomicAdd(d.ctr + CTR_POOL_TOP, 1);
                if (f >= d.n_frames) {
                    atomicOr(d.ctr + CTR_ERROR, PIC_DEV_FRAME_POOL_EXHAUSTED);
                    d.sc_nframes[s] = i;
                    return;
                }
            }
            d.tbl_pool[off + i] = f;
        }
        d.sc_nframes[s] = need;
    }
    d.sc_tail[s] = count;
    d.sc_incoming[s] = 0;
    const int next = (d.nosort ? d.sc_next[s] : count) - d.sc_left[s] + inc;
    d.sc_next[s] = next;                            // population after the pending sort
    int listed = 0;
    if (next >= d.crowd_min) {                      // crowded: the next step starts it first (pic_cta_supercell)
        const int at = atomicAdd(d.ctr + CTR_CROWD, 1);
        if (at < PIC_CROWD_MAX) {
            d.crowd_list[at] = s;
            listed = 1;
        }
    }
    d.sc_crowd[s] = listed;
    d.sc_left[s] = 0;
    // (largest population seen: particles, not slots — after a step without a sort `count` includes the holes)
    atomicMax(d.ctr + CTR_MAX_COUNT, (d.nosort ? next : count + inc));
    if (next > 0) atomicMax(d.ctr + CTR_NEGMIN, (1 << 30) - next);
    // how many supercells fall on either side of the sparse/dense line (one atomic per warp and side): the host reads
    // the two counts at its next synchronisation and launches one class of variants only where the other is < 2 %
    {
        const unsigned m = __activemask();              // (threads beyond the last supercell or after a fault have left)
        const unsigned dense = __ballot_sync(m, next >= d.direct_below);
        const unsigned sparse = __ballot_sync(m, next > 0 && next < d.direct_below);
        if ((int)(threadIdx.x & 31) == __ffs(m) - 1) {
            if (dense) atomicAdd(d.ctr + CTR_NDENSE, __popc(dense));
            if (sparse) atomicAdd(d.ctr + CTR_NSPARSE, __popc(sparse));
        }
    }
}

// Table regions abandoned by the pic_prepare_kernel launched just before go back to the free list of their class
// (push only; the next prepare pops).
__global__ void pic_reclaim_tables_kernel(const PicDev d)
{
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < d.nsc; s += gridDim.x * blockDim.x) {
        const int ocap = d.tbl_old_cap[s];
        if (ocap == 0) continue;
        int k = 3;
        while ((1 << k) < ocap) ++k;
        const int at = atomicAdd(d.tbl_free_top + k, 1);
        if (at < PIC_TBL_FREE) d.tbl_free[k * PIC_TBL_FREE + at] = d.tbl_old_off[s];
        else atomicSub(d.tbl_free_top + k, 1);          // list full: the region is lost (never handed out twice)
        d.tbl_old_cap[s] = 0;
    }
}

// One thread per leaver: claim a slot behind the destination's current slots (pool cur).
__global__ void pic_scatter_kernel(const PicDev d)
{
    const int n = min(d.ctr[CTR_EXCH], d.x_cap);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (d.ctr[CTR_FREE_TOP] < 0) d.ctr[CTR_FREE_TOP] = 0;      // see pic_prepare_kernel
        d.ctr[CTR_LEAVERS_LAST] = n;
        atomicAdd(d.ctr64 + CTR64_LEAVERS_CUM, (unsigned long long)n);
    }
    float4* rec = d.rec[d.cur];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int dst = d.x_dst[i];
        const int slot = atomicAdd(d.sc_tail + dst, 1);
        const int fr = slot >> 8;
        if (fr < d.sc_nframes[dst]) {
            const size_t idx = (size_t)d.tbl_pool[d.tbl_off[dst] + fr] * PIC_FRAME + (slot & (PIC_FRAME - 1));
            rec[2 * idx] = d.x_rec[2 * (size_t)i];
            rec[2 * idx + 1] = d.x_rec[2 * (size_t)i + 1];
            d.pid[d.cur][idx] = d.x_id[i];
        }
    }
}

// One CTA per supercell: counting sort by NEW local cell from pool cur (slots [0,tail): stayers,
// holes of leavers, appended arrivals) into the other pool; publishes the cell ranges, the
// thread->cell assignment of the next step (cells by decreasing count, so that the 32 cells of
// a warp hold similar numbers of particles) and the new count; clears the histogram.
__global__ void __launch_bounds__(PIC_FRAME) pic_sort_kernel(const PicDev d)
{
    __shared__ int s_cnt[256];
    __shared__ int s_cur[256];
    __shared__ int s_wsum[8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int s = blockIdx.x;
    if (d.sort_filter && d.sc_next[s] >= d.direct_below) return;     // a dense step CTA sorts this one itself
    const int n_scan = min(d.sc_tail[s], d.sc_nframes[s] * PIC_FRAME);     // (see fused_sort: never beyond the owned frames)
    if (n_scan == 0) return;       // empty and nothing arrived: ranges, count and histogram are already zero
    const int cnt = d.cell_hist[(size_t)s * 256 + tid];
    d.cell_hist[(size_t)s * 256 + tid] = 0;
    s_cnt[tid] = cnt;
    // exclusive scan of the 256 counts
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) s_wsum[warp] = inc;
    __syncthreads();
    int wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        if (w < warp) wbase += s_wsum[w];
        total += s_wsum[w];
    }
    const int off = wbase + inc - cnt;
    s_cur[tid] = off;
    d.cell_off[(size_t)s * 257 + tid] = off;
    if (tid == 0) {
        d.cell_off[(size_t)s * 257 + 256] = total;
        d.sc_count[s] = total;
    }
    // work items of the next step: cell c is cut into k = ceil(n/T) segments of ~n/k particles; order
    // the cells by decreasing segment length (ties by index) and publish the first item of each
    if (total >= d.direct_below) {   // block-uniform; the per-particle path needs no work items
    const int seg_T = pic_segment_target(total, d.seg_num, d.two_phase ? PIC_ITEM_LMAX(d.order) : 0);
    const int k = (cnt + seg_T - 1) / seg_T;
    const int seglen = k ? (cnt + k - 1) / k : 0;
    __syncthreads();               // s_cnt is complete; reuse it for the keys
    const int key = seglen;
    s_cnt[tid] = key;
    __syncthreads();
    int rank = 0;
    for (int c = 0; c < 256; ++c) {
        const int v = s_cnt[c];
        rank += (v > key) || (v == key && c < tid);
    }
    d.cell_perm[(size_t)s * 256 + rank] = (unsigned char)tid;
    __syncthreads();
    s_cnt[rank] = k;               // segments per cell, in item order
    __syncthreads();
    {
        const int kk = s_cnt[tid];
        int ki = kk;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int v = __shfl_up_sync(0xffffffffu, ki, o);
            if (lane >= o) ki += v;
        }
        __syncthreads();           // s_wsum of the first scan has been read by everyone
        if (lane == 31) s_wsum[warp] = ki;
        __syncthreads();
        int kb = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w)
            if (w < warp) kb += s_wsum[w];
        d.cell_kbase[(size_t)s * 256 + tid] = (unsigned short)min(kb + ki - kk, 65535);
    }
    }
    __syncthreads();
    if (total > n_scan) {          // histogram and records disagree: never write out of bounds
        if (tid == 0) atomicOr(d.ctr + CTR_ERROR, PIC_DEV_SORT_MISMATCH);
        return;
    }
    const int* tbl = d.tbl_pool + d.tbl_off[s];
    const float4* src = d.rec[d.cur];
    float4* dst = d.rec[d.cur ^ 1];
    const uint32_t* sid = d.pid[d.cur];
    uint32_t* did = d.pid[d.cur ^ 1];
    // four slots per thread and iteration: all loads are issued before the first use
    constexpr int U = 4;
    for (int base = 0; base < n_scan; base += U * PIC_FRAME) {
        size_t i[U];
        float4 P[U], M[U];
        uint32_t id[U];
        bool ok[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int slot = base + u * PIC_FRAME + tid;
            ok[u] = slot < n_scan;
            i[u] = ok[u] ? (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1)) : 0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (ok[u]) {
                load_record256(src + 2 * i[u], P[u], M[u]);
                id[u] = sid[i[u]];
            }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (!ok[u]) continue;
            const uint32_t bits = __float_as_uint(M[u].w);
            if (bits & PIC_LEFT_FLAG) continue;
            const int r = atomicAdd(&s_cur[bits & 0xff], 1);
            if (r >= total) {
                atomicOr(d.ctr + CTR_ERROR, PIC_DEV_SORT_MISMATCH);
                continue;
            }
            const size_t o = (size_t)tbl[r >> 8] * PIC_FRAME + (r & (PIC_FRAME - 1));
            store_record256(dst + 2 * o, P[u], M[u]);
            did[o] = id[u];
        }
    }
    // a supercell that shrank returns the frames it no longer needs (one spare is kept); they are
    // free in both pools and are handed out again by the next pic_prepare_kernel
    __syncthreads();
    if (tid == 0) {
        const int keep = (total + PIC_FRAME - 1) / PIC_FRAME + 1, have = d.sc_nframes[s];
        if (have > keep) {
            const int at = atomicAdd(d.ctr + CTR_FREE_TOP, have - keep);
            for (int i = keep; i < have; ++i) d.free_stack[at + i - keep] = tbl[i];
            d.sc_nframes[s] = keep;
        }
    }
}

}  // namespace

template <int O, bool TMA, bool FIX, int MODE>
static cudaError_t launch_step_one(const PicDev& d, const CUtensorMap& map, cudaStream_t st)
{
    static bool configured = false;     // opt in to > 48 KB of dynamic shared memory once
    constexpr bool SPARSE = MODE == PIC_MODE_SPARSE;
    constexpr int bytes = SPARSE ? StepSmem<O, FIX>::OFF_SLOW
                                 : MODE == PIC_MODE_ONE ? StepSmem<O, FIX>::OFF_STGP : StepSmem<O, FIX>::TOTAL;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(pic_step_kernel<O, TMA, FIX, MODE>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        int ctas = 0;                   // the design point is two dense CTAs (three sparse ones) per SM
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, pic_step_kernel<O, TMA, FIX, MODE>,
                                                          SPARSE ? 256 : PIC_STEP_THREADS, bytes);
        if (e != cudaSuccess) return e;
        if (ctas < 2) return cudaErrorLaunchOutOfResources;
        configured = true;
    }
    pic_step_kernel<O, TMA, FIX, MODE><<<pic_step_grid(d), SPARSE ? 256 : PIC_STEP_THREADS, bytes, st>>>(d, map);
    return cudaGetLastError();
}

template <int O, bool TMA, bool FIX>
static cudaError_t launch_step_variant(const PicDev& d, const CUtensorMap& map, cudaStream_t st, int64_t* launches, int cell,
                                       const PicAux& aux)
{
    cudaError_t e = cudaSuccess;
    if (d.class_all != 1 && cell) {     // dense supercells: the whole-cell kernel of pic_cell.cu (fixed point only)
        e = pic_launch_cell(d, O, TMA, &map, st, launches, cell == 2);
    } else if (d.class_all != 1 && d.two_phase && aux.stream) {
        // Both dense variants, side by side: they take disjoint supercells and meet only in atomics (J, the exchange
        // buffer, the frame stack, the counters).  The crowded supercells (one-phase variant: a few hundred CTAs that
        // run for milliseconds and leave SMs idle at their end — profiles/README.md, hot-spot table) are launched first,
        // on the second stream; the ordinary supercells' CTAs fill what they leave free.
        e = cudaEventRecord(aux.fork, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(aux.stream, aux.fork, 0);
        if (e == cudaSuccess) e = launch_step_one<O, TMA, FIX, PIC_MODE_ONE>(d, map, aux.stream);
        if (e == cudaSuccess) e = launch_step_one<O, TMA, FIX, PIC_MODE_TWO>(d, map, st);
        if (e == cudaSuccess) e = cudaEventRecord(aux.join, aux.stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, aux.join, 0);
        *launches += 2;
    } else if (d.class_all != 1) {      // dense variants (none when the host knows every supercell to be sparse)
        if (d.two_phase) {
            e = launch_step_one<O, TMA, FIX, PIC_MODE_TWO>(d, map, st);
            ++*launches;
        }
        if (e == cudaSuccess) {          // crowded supercells (a stale belief must not hide one) / two_phase off
            e = launch_step_one<O, TMA, FIX, PIC_MODE_ONE>(d, map, st);
            ++*launches;
        }
    }
    if (e == cudaSuccess && d.class_all != 2) {
        if (FIX && d.sparse_float_tile) {      // sparse supercells: float shared tile, fixed-point global accumulators
            PicDev ds = d;
            ds.float_tile_to_j64 = 1;
            e = launch_step_one<O, TMA, false, PIC_MODE_SPARSE>(ds, map, st);
        } else {
            e = launch_step_one<O, TMA, FIX, PIC_MODE_SPARSE>(d, map, st);
        }
        ++*launches;
    }
    return e;
}

cudaError_t pic_launch_step(const PicDev& d, int order, bool use_tma, bool fixed_point, const void* tmap,
                            cudaStream_t st, int64_t* launches, int cell_kernel, const PicAux& aux)
{
    const int cell = fixed_point ? cell_kernel : 0;
    CUtensorMap map;
    if (use_tma) memcpy(&map, tmap, sizeof map); else memset(&map, 0, sizeof map);
    cudaError_t e;
#define PIC_GO(O)                                                                               \
    e = use_tma ? (fixed_point ? launch_step_variant<O, true, true>(d, map, st, launches, cell, aux)                 \
                               : launch_step_variant<O, true, false>(d, map, st, launches, cell, aux))               \
                : (fixed_point ? launch_step_variant<O, false, true>(d, map, st, launches, cell, aux)                \
                               : launch_step_variant<O, false, false>(d, map, st, launches, cell, aux))
    switch (order) {
        case 1: PIC_GO(1); break;
        case 2: PIC_GO(2); break;
        default: PIC_GO(3); break;
    }
#undef PIC_GO
    return e;
}

cudaError_t pic_launch_overflow(const PicDev& d, int order, bool fixed_point, cudaStream_t st, int64_t* launches)
{
    const dim3 g(148 * 2), b(128);
    switch (order * 2 + (fixed_point ? 1 : 0)) {
        case 2: pic_overflow_kernel<1, false><<<g, b, 0, st>>>(d); break;
        case 3: pic_overflow_kernel<1, true><<<g, b, 0, st>>>(d); break;
        case 4: pic_overflow_kernel<2, false><<<g, b, 0, st>>>(d); break;
        case 5: pic_overflow_kernel<2, true><<<g, b, 0, st>>>(d); break;
        case 6: pic_overflow_kernel<3, false><<<g, b, 0, st>>>(d); break;
        default: pic_overflow_kernel<3, true><<<g, b, 0, st>>>(d); break;
    }
    ++*launches;
    return cudaGetLastError();
}

__global__ void pic_zero_ints_kernel(int4* p, size_t n16)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
        p[i] = make_int4(0, 0, 0, 0);
}

cudaError_t pic_launch_zero_ints(int* p, size_t n, cudaStream_t st, int64_t* launches)
{
    pic_zero_ints_kernel<<<148 * 8, 256, 0, st>>>(reinterpret_cast<int4*>(p), n / 4);     // n is a multiple of 256
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pic_launch_convert(const PicDev& d, cudaStream_t st, int64_t* launches)
{
    pic_convert_J_kernel<<<148 * 8, 256, 0, st>>>(d);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pic_launch_prepare(const PicDev& d, cudaStream_t st, int64_t* launches)
{
    cudaError_t e0 = cudaMemsetAsync(d.ctr + CTR_CROWD, 0, 3 * sizeof(int), st);  // crowd list and the two class counts (CTR_CROWD, CTR_NDENSE, CTR_NSPARSE are adjacent) are rebuilt by every prepare
    if (e0 != cudaSuccess) return e0;
    pic_prepare_kernel<<<(d.nsc + 255) / 256, 256, 0, st>>>(d);
    pic_reclaim_tables_kernel<<<(d.nsc + 255) / 256, 256, 0, st>>>(d);
    *launches += 2;
    return cudaGetLastError();
}

cudaError_t pic_launch_scatter(const PicDev& d, cudaStream_t st, int64_t* launches)
{
    pic_scatter_kernel<<<148 * 4, 256, 0, st>>>(d);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t pic_launch_sort(const PicDev& d, cudaStream_t st, int64_t* launches)
{
    pic_sort_kernel<<<d.nsc, PIC_FRAME, 0, st>>>(d);
    ++*launches;
    return cudaGetLastError();
}
