// pic_api.cu — the C ABI of include/pic_b200.h: context, workspace carving, particle
// load / read-back, field upload.  The step itself is in pic_step.cu.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <cuda.h>

#include <new>
#include <string>
#include <vector>

#include "../../include/pic_b200.h"
#include "pic_internal.cuh"

struct pic_ctx {
    PicDev d;
    int order;
    double cell[3], dt;
    double q[PIC_NSPECIES], m[PIC_NSPECIES];
    int n_species;               // slots set by pic_set_species (PIC_NSPECIES while the defaults q=-1, m=1 stand)
    int64_t max_particles, n_particles, steps, launches;
    cudaStream_t stream;
    bool have_fields;
    bool use_tma, fixed_point;
    int cell_kernel;             // option "cell_kernel": dense supercells go to 0 the round-1 kernels, 1 pic_cell_kernel, 2 the persistent pic_pcell_kernel
    bool fuse_sort;              // option "fuse_sort": the step kernel sorts its supercell first (default on)
    bool field_update;           // option "field_update": every step ends with a Yee update of E, B (pic_fields.cu)
    float* Fbuf[2];              // the two PADDED field buffers (periodic halos pre-filled); d.Fpad == Fbuf[F_cur]
    int F_cur;
    bool yee_index64;            // option "yee_index64": force the 64-bit-index instantiation (taken anyway beyond 2^32 elements)
    int yee_tile;                // option "yee_tile": y extent of the Yee kernel's tile (8 or 16; 0 = the measured best)
    PicAux aux;                  // second stream for the crowded supercells' variant (option "overlap"), with its events
    bool overlap;
    bool yee_wide;               // option "yee_wide": four cells per thread where the grid is at least 64 wide (default)
    bool dirty;                  // pool cur holds a stepped state whose sort is still pending
    bool sparse_nosort;          // option "sparse_nosort": all-sparse steps skip the re-sort (default on)
    int nosort_period;           // ... and one step in this many sorts
    int steps_unsorted;          // steps since the last sort
    bool sparse_float;           // option "sparse_float": all-sparse steps deposit in float (default on)
    int crowd_min_on;            // PicDev::crowd_min when option "crowd_first" is on
    int force_class;             // option "class_all": -1 = from the counters (default), 0/1/2 = PicDev::class_all as given
    int n_dense, n_sparse;       // non-empty supercells on either side of the sparse/dense line at the last synchronisation
    int max_known, min_known;    // largest / smallest non-empty supercell population as of the last synchronisation (0: unknown)
    int* hist[2];                // the two cell histograms; d.cell_hist == hist[hist_cur]
    int hist_cur;
    char* ws;
    uint64_t ws_bytes;
    std::string err;
    // TMA descriptor of the padded field copy
    alignas(64) unsigned char tmap[2][128];     // one tensor map per padded buffer
    bool tmap_ok;
    // option "timing": CUDA events around every launch of the step kernel
    bool timing;
    std::vector<cudaEvent_t> events;
};

// all-sparse steps: one sort in this many steps by default (option "sparse_nosort" >= 2 sets another period).  Measured on
// configs[2], average over its 50 steps: 8 -> 5.91 ms per step, 16 -> 5.77, 32 -> 5.74 (a sort costs 2.7 ms; the
// unsorted steps slow down by 0.3 ms over 25 steps as holes and disorder grow)
#define PIC_NOSORT_PERIOD 16

static std::string g_create_error;

// ------------------------------------------------------------------ workspace layout
namespace {

struct Layout {
    uint64_t rec0, rec1, pid0, pid1, free_stack, tbl_pool, tbl_off, tbl_cap, tbl_old_off, tbl_old_cap, tbl_free, tbl_free_top, sc_nframes, sc_count, sc_tail, sc_incoming,
        sc_left, sc_next, sc_crowd, crowd_list, cell_off, cell_hist, cell_perm, cell_kbase, x_rec, x_id, x_dst, ovf, ctr, ctr64, Fpad, Fpad2, J, J64, sc_offset, total;
    int n_frames, tbl_pool_size, x_cap, nsc;
};

uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

int compute_layout(const int32_t grid[3], const int32_t sc[3], int order, int64_t maxp, Layout* L)
{
    if (!grid || !sc) return PIC_EINVAL;
    if (sc[0] != PIC_SCX || sc[1] != PIC_SCY || sc[2] != PIC_SCZ) return PIC_EINVAL;
    if (order < 1 || order > 3 || maxp < 0) return PIC_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (grid[a] <= 0 || grid[a] % sc[a] != 0) return PIC_EINVAL;
    const uint64_t nsc = (uint64_t)(grid[0] / sc[0]) * (grid[1] / sc[1]) * (grid[2] / sc[2]);
    const uint64_t ncell = (uint64_t)grid[0] * grid[1] * grid[2];
    if (nsc > (1u << 22) || (uint64_t)maxp > (1ull << 32) - 1) return PIC_EINVAL;   // supercell index is packed into 23 bits
    // every supercell may hold one partly filled frame; 1/8 head-room for density drift
    const uint64_t n_frames = (uint64_t)maxp / PIC_FRAME + (uint64_t)maxp / (8 * PIC_FRAME) + 2 * nsc + 64;
    const uint64_t slots = n_frames * PIC_FRAME;
    const uint64_t tblp = 4 * n_frames + 16 * nsc + 1024;
    uint64_t xcap = (uint64_t)maxp / 4 + 65536;
    if (xcap > (uint64_t)maxp + 1024) xcap = (uint64_t)maxp + 1024;
    if (n_frames > 0x7fffffffull / 2 || tblp > 0x7fffffffull || xcap > 0x7fffffffull) return PIC_EINVAL;
    uint64_t o = 0;
    auto take = [&](uint64_t bytes) { uint64_t r = o; o = align_up(o + bytes, 256); return r; };
    L->rec0 = take(slots * 32);
    L->rec1 = take(slots * 32);
    L->pid0 = take(slots * 4);
    L->pid1 = take(slots * 4);
    L->free_stack = take(n_frames * 4);
    L->tbl_pool = take(tblp * 4);
    L->tbl_off = take(nsc * 4);
    L->tbl_cap = take(nsc * 4);
    L->tbl_old_off = take(nsc * 4);
    L->tbl_old_cap = take(nsc * 4);
    L->tbl_free = take((uint64_t)PIC_TBL_CLASSES * PIC_TBL_FREE * 4);
    L->tbl_free_top = take(PIC_TBL_CLASSES * 4);
    L->sc_nframes = take(nsc * 4);
    L->sc_count = take(nsc * 4);
    L->sc_tail = take(nsc * 4);
    L->sc_incoming = take(nsc * 4);
    L->sc_left = take(nsc * 4);
    L->sc_next = take(nsc * 4);
    L->sc_crowd = take(nsc * 4);
    L->crowd_list = take(PIC_CROWD_MAX * 4);
    L->cell_off = take(nsc * 257 * 4);
    L->cell_hist = take(2 * nsc * 256 * 4);      // two histograms (this step's, the previous step's)
    L->cell_perm = take(nsc * 256);
    L->cell_kbase = take(nsc * 256 * 2);
    L->x_rec = take(xcap * 32);
    L->x_id = take(xcap * 4);
    L->x_dst = take(xcap * 4);
    L->ovf = take(xcap * 32);
    L->ctr = take(CTR_N * 4);
    L->ctr64 = take(CTR64_N * 8);
    // the fields live in PADDED arrays only (what the step kernel's TMA reads); two of them: the Yee update reads level
    // n from one and writes level n+1, every periodic image included, to the other
    const uint64_t npad6 = 6ull * (grid[0] + PIC_PAD_X) * (grid[1] + PIC_PAD_Y) * (grid[2] + PIC_PAD_Z) * 4;
    L->Fpad = take(npad6);
    L->Fpad2 = take(npad6);
    L->J = take(3 * ncell * 4);
    L->J64 = take(3 * ncell * 8);
    L->sc_offset = take((nsc + 1) * 8);
    L->total = o;
    L->n_frames = (int)n_frames;
    L->tbl_pool_size = (int)tblp;
    L->x_cap = (int)xcap;
    L->nsc = (int)nsc;
    return PIC_OK;
}

int fail(pic_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

int cuda_fail(pic_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, PIC_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// ------------------------------------------------------------------ load kernels
// Position (float64, physical units) -> wrapped integer cell + fp32 in-cell fraction.
__device__ __forceinline__ void split_position(double x, double inv_cell, int n, int& cell, float& frac)
{
    double X = x * inv_cell;
    double c = floor(X);
    float f = (float)(X - c);
    if (f >= 1.0f) { f = 0.0f; c += 1.0; }
    if (f < 0.0f) f = 0.0f;
    double r = fmod(c, (double)n);
    if (r < 0) r += (double)n;
    cell = (int)r;
    if (cell >= n) cell = 0;
    frac = f;
}

struct LoadArgs {
    const double *x, *y, *z;
    const float *ux, *uy, *uz, *w;
    const int32_t* species;
    long long n;
    unsigned id0;
    double icx, icy, icz;
};

__device__ __forceinline__ int load_locate(const PicDev& d, const LoadArgs& a, long long i,
                                           float4& P, int& lc)
{
    int cx, cy, cz;
    float fx, fy, fz;
    split_position(a.x[i], a.icx, d.nx, cx, fx);
    split_position(a.y[i], a.icy, d.ny, cy, fy);
    split_position(a.z[i], a.icz, d.nz, cz, fz);
    P = make_float4(fx, fy, fz, a.w[i]);
    lc = (cx % PIC_SCX) + PIC_SCX * ((cy % PIC_SCY) + PIC_SCY * (cz % PIC_SCZ));
    return (cx / PIC_SCX) + d.nsx * ((cy / PIC_SCY) + d.nsy * (cz / PIC_SCZ));
}

__global__ void pic_load_count_kernel(const PicDev d, const LoadArgs a)
{
    int wmax = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.n;
         i += (long long)gridDim.x * blockDim.x) {
        float4 P;
        int lc;
        int s = load_locate(d, a, i, P, lc);
        atomicAdd(d.sc_incoming + s, 1);
        atomicAdd(d.cell_hist + (size_t)s * 256 + lc, 1);
        wmax = max(wmax, __float_as_int(fabsf(a.w[i])));
        if (a.species && (a.species[i] < 0 || a.species[i] >= d.n_species)) atomicOr(d.ctr + CTR_ERROR, PIC_DEV_BAD_SPECIES);
    }
    // one atomic per warp, and only if it raises the maximum (a per-particle atomicMax on one address
    // serialises in L2: 0.8 ms per 8 M particles)
    wmax = __reduce_max_sync(0xffffffffu, wmax);
    if ((threadIdx.x & 31) == 0 && wmax > d.ctr[CTR_WMAX_BITS]) atomicMax(d.ctr + CTR_WMAX_BITS, wmax);
}

__global__ void pic_load_scatter_kernel(const PicDev d, const LoadArgs a)
{
    if (blockIdx.x == 0 && threadIdx.x == 0 && d.ctr[CTR_FREE_TOP] < 0) d.ctr[CTR_FREE_TOP] = 0;   // see pic_prepare_kernel
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.n;
         i += (long long)gridDim.x * blockDim.x) {
        float4 P;
        int lc;
        const int s = load_locate(d, a, i, P, lc);
        const int sp = a.species ? a.species[i] : 0;
        const int slot = atomicAdd(d.sc_tail + s, 1);
        const int fr = slot >> 8;
        if (fr < d.sc_nframes[s]) {
            const size_t idx = (size_t)d.tbl_pool[d.tbl_off[s] + fr] * PIC_FRAME + (slot & (PIC_FRAME - 1));
            d.rec[d.cur][2 * idx] = P;
            d.rec[d.cur][2 * idx + 1] = make_float4(a.ux[i], a.uy[i], a.uz[i],
                                                    __uint_as_float(pic_pack_bits(lc, sp & (PIC_NSPECIES - 1))));
            d.pid[d.cur][idx] = a.id0 + (unsigned)i;
        }
    }
}

// Before an appending load is sorted in: count the particles already present per cell.
__global__ void pic_hist_add_present_kernel(const PicDev d)
{
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= (size_t)d.nsc * 256) return;
    const size_t s = i >> 8, c = i & 255;
    d.cell_hist[i] += d.cell_off[s * 257 + c + 1] - d.cell_off[s * 257 + c];
}

// ------------------------------------------------------------------ read-back kernels
__global__ void pic_scan_counts_kernel(const PicDev d)
{
    __shared__ long long part[1024];
    const int t = threadIdx.x;
    const int per = (d.nsc + 1023) / 1024;
    const int lo = min(t * per, d.nsc), hi = min(lo + per, d.nsc);
    long long sum = 0;
    for (int i = lo; i < hi; ++i) sum += d.sc_count[i];
    part[t] = sum;
    __syncthreads();
    if (t == 0) {
        long long run = 0;
        for (int i = 0; i < 1024; ++i) { long long v = part[i]; part[i] = run; run += v; }
        d.sc_offset[d.nsc] = run;
    }
    __syncthreads();
    long long run = part[t];
    for (int i = lo; i < hi; ++i) { d.sc_offset[i] = run; run += d.sc_count[i]; }
}

struct GetArgs {
    double *x, *y, *z;
    float *ux, *uy, *uz, *w;
    int32_t* species;
    uint32_t* id;
    int32_t* supercell;
    long long capacity;
    double cx, cy, cz;
};

__global__ void pic_get_particles_kernel(const PicDev d, const GetArgs a)
{
    const int s = blockIdx.x;
    const int count = d.sc_count[s];
    const long long off = d.sc_offset[s];
    const int* tbl = d.tbl_pool + d.tbl_off[s];
    const int ox = (s % d.nsx) * PIC_SCX, oy = ((s / d.nsx) % d.nsy) * PIC_SCY, oz = (s / (d.nsx * d.nsy)) * PIC_SCZ;
    for (int slot = threadIdx.x; slot < count; slot += blockDim.x) {
        const long long o = off + slot;
        if (o >= a.capacity) break;
        const size_t idx = (size_t)tbl[slot >> 8] * PIC_FRAME + (slot & (PIC_FRAME - 1));
        const float4 P = d.rec[d.cur][2 * idx];
        const float4 M = d.rec[d.cur][2 * idx + 1];
        const uint32_t bits = __float_as_uint(M.w);
        const int lc = bits & 0xffff;
        if (a.x) a.x[o] = ((double)(ox + (lc & 7)) + (double)P.x) * a.cx;
        if (a.y) a.y[o] = ((double)(oy + ((lc >> 3) & 7)) + (double)P.y) * a.cy;
        if (a.z) a.z[o] = ((double)(oz + (lc >> 6)) + (double)P.z) * a.cz;
        if (a.ux) a.ux[o] = M.x;
        if (a.uy) a.uy[o] = M.y;
        if (a.uz) a.uz[o] = M.z;
        if (a.w) a.w[o] = P.w;
        if (a.species) a.species[o] = (bits >> 16) & 0xff;
        if (a.id) a.id[o] = d.pid[d.cur][idx];
        if (a.supercell) a.supercell[o] = s;
    }
}

// Caller's plain arrays -> padded array with periodic halos (the only form the fields are kept in), and back.
struct FieldPtrs { const float* src[6]; float* dst[6]; };

// A CTA takes PIC_PADROWS consecutive rows (one per warp at a time) of one plane of one component of the padded
// (pad) or plain (unpad) array: component, plane and wraps are worked out per CTA and per row, the lanes run along x.
// (An index decomposition per element, with 64-bit divisions by run-time extents, took 3.4 ms on the 67 M-cell grid;
// one CTA per row 2.6 ms: 1.6 M CTAs of 1 KB each.)
#define PIC_PADROWS 32

__global__ void pic_pad_fields_kernel(const PicDev d, const FieldPtrs f, float* pad)
{
    const int px = d.nx + PIC_PAD_X, py = d.ny + PIC_PAD_Y, pz = d.nz + PIC_PAD_Z;
    const int nchunk = (py + PIC_PADROWS - 1) / PIC_PADROWS;
    int b = blockIdx.x;                            // (c, k, chunk of rows) of the padded array
    const int j0 = (b % nchunk) * PIC_PADROWS; b /= nchunk;
    const int k = b % pz;
    const int c = b / pz;
    const int gk = ((k - PIC_PAD_LO) % d.nz + d.nz) % d.nz;
    const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    for (int j = j0 + (threadIdx.x >> 5); j < min(j0 + PIC_PADROWS, py); j += nwarp) {
        const int gj = ((j - PIC_PAD_LO) % d.ny + d.ny) % d.ny;
        const float* src = f.src[c] + (size_t)d.nx * ((size_t)gj + (size_t)d.ny * gk);
        float* dst = pad + (size_t)px * ((size_t)j + (size_t)py * ((size_t)k + (size_t)pz * c));
        for (int i = lane; i < px; i += 32) {
            int gi = i - d.pad_lo_x;
            if (gi < 0) gi = (gi % d.nx + d.nx) % d.nx;
            else if (gi >= d.nx) gi %= d.nx;
            dst[i] = src[gi];
        }
    }
}

__global__ void pic_unpad_fields_kernel(const PicDev d, const FieldPtrs f, const float* pad)
{
    const int px = d.nx + PIC_PAD_X, py = d.ny + PIC_PAD_Y, pz = d.nz + PIC_PAD_Z;
    const int nchunk = (d.ny + PIC_PADROWS - 1) / PIC_PADROWS;
    int b = blockIdx.x;                            // (c, k, chunk of rows) of the plain arrays
    const int j0 = (b % nchunk) * PIC_PADROWS; b /= nchunk;
    const int k = b % d.nz;
    const int c = b / d.nz;
    if (!f.dst[c]) return;
    const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    for (int j = j0 + (threadIdx.x >> 5); j < min(j0 + PIC_PADROWS, d.ny); j += nwarp) {
        const float* src = pad + (size_t)d.pad_lo_x + (size_t)px * ((size_t)(j + PIC_PAD_LO) + (size_t)py * ((size_t)(k + PIC_PAD_LO) + (size_t)pz * c));
        float* dst = f.dst[c] + (size_t)d.nx * ((size_t)j + (size_t)d.ny * k);
        for (int i = lane; i < d.nx; i += 32) dst[i] = src[i];
    }
}

void refresh_species(pic_ctx* c)
{
    for (int s = 0; s < PIC_NSPECIES; ++s) {
        c->d.h[s] = (float)((c->q[s] / c->m[s]) * c->dt * 0.5);
        c->d.q[s] = (float)c->q[s];
    }
    // the fixed-point scale of J follows max|q| over the slots in use only: the default q = -1 of slots the caller
    // never set must not pin it when the table holds physical charges
    double qmax = 0.0;
    for (int s = 0; s < c->n_species; ++s) qmax = fmax(qmax, fabs(c->q[s]));
    c->d.qmax = (float)qmax;
    c->d.n_species = c->n_species;
}

// explicit Yee scheme: stable for c*dt*sqrt(1/dx^2 + 1/dy^2 + 1/dz^2) < 1 (the particle step alone only needs c*dt < cell)
bool yee_stable(const pic_ctx* c)
{
    double s = 0.0;
    for (int a = 0; a < 3; ++a) s += 1.0 / (c->cell[a] * c->cell[a]);
    return c->dt * sqrt(s) < 1.0;
}

int check_device(pic_ctx* c)
{
    int ctr[CTR_N] = {0};
    cudaError_t e = cudaMemcpyAsync(ctr, c->d.ctr, sizeof ctr, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "reading the device error word");
    const int err = ctr[CTR_ERROR];
    // populations seen so far (running max / min): lets the next steps skip kernel variants no supercell needs
    c->max_known = ctr[CTR_MAX_COUNT];
    c->n_dense = ctr[CTR_NDENSE];
    c->n_sparse = ctr[CTR_NSPARSE];
    c->min_known = ctr[CTR_NEGMIN] ? (1 << 30) - ctr[CTR_NEGMIN] : 0;
    if (err) {
        char buf[220];
        snprintf(buf, sizeof buf, "device fault word 0x%x (1 frame pool, 2 exchange buffer, 4 table pool, 8 moved >= 1 cell, 16 TMA timeout, 32 overflow queue, 64 sort mismatch, 128 species id outside the table)", err);
        return fail(c, PIC_EDEVICE, buf);
    }
    return PIC_OK;
}

}  // namespace

// 4-D tensor map (x, y, z, component) over the padded field copy; the step kernel
// fetches a supercell's whole E/B tile with one cp.async.bulk.tensor.
// cuTensorMapEncodeTiled is resolved through the runtime, so libcuda is not a link dependency.
static int pic_build_tensor_map(pic_ctx* c, int which)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(c, PIC_ECUDA, "cuTensorMapEncodeTiled not available");
    }
    const PicDev& d = c->d;
    const int O = c->order;
    const cuuint32_t fn_xy = (O == 1) ? 10 : (O == 2) ? 11 : 12;
    const cuuint64_t px = d.nx + PIC_PAD_X, py = d.ny + PIC_PAD_Y, pz = d.nz + PIC_PAD_Z;
    const cuuint64_t dims[4] = {px, py, pz, 6};
    const cuuint64_t strides[3] = {px * 4, px * py * 4, px * py * pz * 4};
    const cuuint32_t box[4] = {12, fn_xy, fn_xy - (PIC_SCX - PIC_SCZ), 6};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((encode_fn)fn)((CUtensorMap*)c->tmap[which], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)c->Fbuf[which], dims,
                                 strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, PIC_ECUDA, "cuTensorMapEncodeTiled failed");
    return PIC_OK;
}

// ------------------------------------------------------------------ C ABI
extern "C" {

int32_t pic_workspace_bytes(const int32_t grid[3], const int32_t supercell[3], int32_t shape_order,
                            int64_t max_particles, uint64_t* bytes_out)
{
    Layout L;
    int rc = compute_layout(grid, supercell, shape_order, max_particles, &L);
    if (rc != PIC_OK) return fail(nullptr, rc, "pic_workspace_bytes: bad geometry (grid must be a positive multiple of the 8x8x4 supercell, order in 1..3)");
    if (!bytes_out) return fail(nullptr, PIC_EINVAL, "pic_workspace_bytes: bytes_out is NULL");
    *bytes_out = L.total;
    return PIC_OK;
}

int32_t pic_create(pic_ctx** out, const int32_t grid[3], const double cell[3], double dt,
                   const int32_t supercell[3], int32_t shape_order, int64_t max_particles,
                   void* workspace, uint64_t workspace_bytes, void* stream)
{
    if (!out) return fail(nullptr, PIC_EINVAL, "pic_create: out is NULL");
    *out = nullptr;
    Layout L;
    int rc = compute_layout(grid, supercell, shape_order, max_particles, &L);
    if (rc != PIC_OK) return fail(nullptr, rc, "pic_create: bad geometry (grid must be a positive multiple of the 8x8x4 supercell, order in 1..3)");
    if (!cell || !(dt > 0.0)) return fail(nullptr, PIC_EINVAL, "pic_create: cell is NULL or dt <= 0");
    for (int a = 0; a < 3; ++a)
        if (!(cell[a] > 0.0) || !(dt < cell[a]))
            return fail(nullptr, PIC_EINVAL, "pic_create: need cell > 0 and c*dt < cell on every axis");
    if (!workspace || ((uintptr_t)workspace & 255)) return fail(nullptr, PIC_EINVAL, "pic_create: workspace is NULL or not 256-byte aligned");
    if (workspace_bytes < L.total) return fail(nullptr, PIC_ENOMEM, "pic_create: workspace smaller than pic_workspace_bytes()");

    pic_ctx* c = new (std::nothrow) pic_ctx();
    if (!c) return fail(nullptr, PIC_ENOMEM, "pic_create: host allocation failed");
    c->order = shape_order;
    c->dt = dt;
    for (int a = 0; a < 3; ++a) c->cell[a] = cell[a];
    for (int s = 0; s < PIC_NSPECIES; ++s) { c->q[s] = -1.0; c->m[s] = 1.0; }
    c->n_species = PIC_NSPECIES;
    c->max_particles = max_particles;
    c->n_particles = 0;
    c->steps = 0;
    c->launches = 0;
    c->stream = (cudaStream_t)stream;
    c->have_fields = false;
    c->use_tma = true;
    c->fuse_sort = true;
    c->cell_kernel = 0;
    c->sparse_float = true;
    c->sparse_nosort = true;
    c->nosort_period = PIC_NOSORT_PERIOD;
    c->steps_unsorted = 0;
    c->field_update = false;
    c->yee_tile = 0;
    c->aux = PicAux{nullptr, nullptr, nullptr};
    c->overlap = true;
    c->yee_wide = true;
    c->yee_index64 = false;
    c->dirty = false;
    c->max_known = c->min_known = 0;
    c->n_dense = c->n_sparse = 0;
    c->force_class = -1;
    c->fixed_point = true;
    c->tmap_ok = false;
    c->timing = false;
    c->ws = (char*)workspace;
    c->ws_bytes = workspace_bytes;

    PicDev& d = c->d;
    d.nx = grid[0]; d.ny = grid[1]; d.nz = grid[2];
    d.nsx = grid[0] / PIC_SCX; d.nsy = grid[1] / PIC_SCY; d.nsz = grid[2] / PIC_SCZ;
    d.nsc = L.nsc;
    d.dtdx = (float)(dt / cell[0]); d.dtdy = (float)(dt / cell[1]); d.dtdz = (float)(dt / cell[2]);
    const double V = cell[0] * cell[1] * cell[2];
    d.jfx = (float)(cell[0] / dt / V); d.jfy = (float)(cell[1] / dt / V); d.jfz = (float)(cell[2] / dt / V);
    refresh_species(c);
    char* w = c->ws;
    d.rec[0] = (float4*)(w + L.rec0); d.rec[1] = (float4*)(w + L.rec1);
    d.pid[0] = (uint32_t*)(w + L.pid0); d.pid[1] = (uint32_t*)(w + L.pid1);
    d.cur = 0;
    d.seg_num = 3;
    d.two_phase = 1;
    d.order = shape_order;
    d.n_frames = L.n_frames;
    d.free_stack = (int*)(w + L.free_stack);
    d.tbl_pool = (int*)(w + L.tbl_pool); d.tbl_pool_size = L.tbl_pool_size;
    d.tbl_off = (int*)(w + L.tbl_off); d.tbl_cap = (int*)(w + L.tbl_cap);
    d.tbl_old_off = (int*)(w + L.tbl_old_off); d.tbl_old_cap = (int*)(w + L.tbl_old_cap);
    d.tbl_free = (int*)(w + L.tbl_free); d.tbl_free_top = (int*)(w + L.tbl_free_top);
    d.sc_nframes = (int*)(w + L.sc_nframes); d.sc_count = (int*)(w + L.sc_count);
    d.sc_tail = (int*)(w + L.sc_tail); d.sc_incoming = (int*)(w + L.sc_incoming);
    d.sc_left = (int*)(w + L.sc_left); d.sc_next = (int*)(w + L.sc_next);
    d.sc_crowd = (int*)(w + L.sc_crowd); d.crowd_list = (int*)(w + L.crowd_list);
    // crowded-first scheduling (option "crowd_first", off: measured slower): crowded = at least four times
    // the mean population the context was sized for (and not below 8192)
    {
        const int64_t mean4 = 4 * (max_particles / (int64_t)L.nsc);
        c->crowd_min_on = (int)(mean4 > 8192 ? (mean4 < (1 << 30) ? mean4 : (1 << 30)) : 8192);
        d.crowd_min = 1 << 30;
        d.direct_below = PIC_DIRECT_BELOW;
        d.gather_ec = 0;
        d.rest_skip = 1;
        d.nosort = 0;
        d.sparse_float_tile = 0;
        d.float_tile_to_j64 = 0;
    }
    d.fused = 0;
    d.class_all = 0;
    d.sort_filter = 0;
    d.cell_off = (int*)(w + L.cell_off);
    c->hist[0] = (int*)(w + L.cell_hist); c->hist[1] = c->hist[0] + (size_t)L.nsc * 256;
    c->hist_cur = 0;
    d.cell_hist = c->hist[0]; d.cell_hist_prev = c->hist[1];
    d.cell_perm = (unsigned char*)(w + L.cell_perm);
    d.cell_kbase = (unsigned short*)(w + L.cell_kbase);
    d.x_rec = (float4*)(w + L.x_rec);
    d.ovf = (float4*)(w + L.ovf); d.ovf_cap = L.x_cap;
    d.x_id = (uint32_t*)(w + L.x_id); d.x_dst = (int*)(w + L.x_dst); d.x_cap = L.x_cap;
    d.ctr = (int*)(w + L.ctr); d.ctr64 = (unsigned long long*)(w + L.ctr64);
    c->Fbuf[0] = (float*)(w + L.Fpad); c->Fbuf[1] = (float*)(w + L.Fpad2); c->F_cur = 0;
    d.Fpad = c->Fbuf[0]; d.J = (float*)(w + L.J); d.J64 = (long long*)(w + L.J64);
    d.sc_offset = (long long*)(w + L.sc_offset);
    d.pad_lo_x = (shape_order == 3) ? 2 : 1;

    // zero the bookkeeping region [tbl_off, x_rec) and the counters, J
    cudaError_t e = cudaMemsetAsync(w + L.tbl_off, 0, L.x_rec - L.tbl_off, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(w + L.ctr, 0, L.Fpad - L.ctr, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(w + L.J, 0, L.sc_offset - L.J, c->stream);
    if (e != cudaSuccess) { int r = cuda_fail(nullptr, e, "pic_create: cudaMemsetAsync"); delete c; return r; }
    // second stream for the crowded supercells' variant; without it the variants run one after the other
    if (cudaStreamCreateWithFlags(&c->aux.stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->aux.fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->aux.join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        if (c->aux.fork) cudaEventDestroy(c->aux.fork);
        if (c->aux.stream) cudaStreamDestroy(c->aux.stream);
        c->aux = PicAux{nullptr, nullptr, nullptr};
    }
    *out = c;
    return PIC_OK;
}

int32_t pic_set_species(pic_ctx* c, int32_t n, const double* q, const double* m)
{
    if (!c) return PIC_EINVAL;
    if (n < 0 || n > PIC_MAX_SPECIES || !q || !m) return fail(c, PIC_EINVAL, "pic_set_species: n out of range or NULL table");
    for (int s = 0; s < n; ++s) {
        if (!(m[s] > 0.0)) return fail(c, PIC_EINVAL, "pic_set_species: mass must be positive");
        c->q[s] = q[s]; c->m[s] = m[s];
    }
    if (n > 0) c->n_species = n;      // particles of a species id >= n raise PIC_DEV_BAD_SPECIES when loaded
    refresh_species(c);
    return PIC_OK;
}

static int ensure_sorted(pic_ctx* c);

int32_t pic_load_particles(pic_ctx* c, int64_t n, const double* x, const double* y, const double* z,
                           const float* ux, const float* uy, const float* uz, const float* w,
                           const int32_t* species)
{
    if (!c) return PIC_EINVAL;
    if (n < 0) return fail(c, PIC_EINVAL, "pic_load_particles: n < 0");
    if (n == 0) return PIC_OK;
    if (!x || !y || !z || !ux || !uy || !uz || !w) return fail(c, PIC_EINVAL, "pic_load_particles: NULL array");
    if (c->n_particles + n > c->max_particles) return fail(c, PIC_ENOMEM, "pic_load_particles: exceeds max_particles");
    {
        int rc = ensure_sorted(c);
        if (rc != PIC_OK) return rc;
    }
    LoadArgs a;
    a.x = x; a.y = y; a.z = z; a.ux = ux; a.uy = uy; a.uz = uz; a.w = w; a.species = species;
    a.n = n; a.id0 = (unsigned)c->n_particles;
    a.icx = 1.0 / c->cell[0]; a.icy = 1.0 / c->cell[1]; a.icz = 1.0 / c->cell[2];
    const PicDev& d = c->d;
    const int grid = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    // count per supercell and per cell (new + already present), make room, append, sort in
    pic_load_count_kernel<<<grid, 256, 0, c->stream>>>(d, a);
    pic_hist_add_present_kernel<<<(unsigned)(((size_t)d.nsc * 256 + 255) / 256), 256, 0, c->stream>>>(d);
    c->launches += 2;
    cudaError_t e = pic_launch_prepare(d, c->stream, &c->launches);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_load_particles: prepare");
    pic_load_scatter_kernel<<<grid, 256, 0, c->stream>>>(d, a);
    c->launches += 1;
    e = cudaGetLastError();
    if (e == cudaSuccess) e = pic_launch_sort(d, c->stream, &c->launches);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_load_particles: scatter/sort");
    c->d.cur ^= 1;
    c->n_particles += n;
    return PIC_OK;
}

int32_t pic_set_fields(pic_ctx* c, const float* Ex, const float* Ey, const float* Ez,
                       const float* Bx, const float* By, const float* Bz)
{
    if (!c) return PIC_EINVAL;
    FieldPtrs f = {{Ex, Ey, Ez, Bx, By, Bz}, {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr}};
    for (int k = 0; k < 6; ++k)
        if (!f.src[k]) return fail(c, PIC_EINVAL, "pic_set_fields: NULL component");
    pic_pad_fields_kernel<<<6u * (unsigned)((c->d.ny + PIC_PAD_Y + PIC_PADROWS - 1) / PIC_PADROWS) * (unsigned)(c->d.nz + PIC_PAD_Z), 256, 0,
                            c->stream>>>(c->d, f, c->Fbuf[c->F_cur]);
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_set_fields: pad kernel");
    if (!c->tmap_ok) c->tmap_ok = (pic_build_tensor_map(c, 0) == PIC_OK && pic_build_tensor_map(c, 1) == PIC_OK);
    c->have_fields = true;
    return PIC_OK;
}

// Sort the supercells of a stepped state (holes of leavers, appended arrivals) into the other pool.
static int ensure_sorted(pic_ctx* c)
{
    if (!c->dirty) return PIC_OK;
    c->d.fused = 0;
    c->d.nosort = 0;
    c->steps_unsorted = 0;
    cudaError_t e = pic_launch_sort(c->d, c->stream, &c->launches);
    if (e != cudaSuccess) return cuda_fail(c, e, "sort");
    c->d.cur ^= 1;
    c->dirty = false;
    return PIC_OK;
}

// One Yee update with the last step's J: level n in the padded buffer Fbuf[F_cur] -> level n+1 in the other one.
static cudaError_t enqueue_field_update(pic_ctx* c, cudaStream_t st)
{
    cudaError_t e = pic_launch_yee(c->d, c->Fbuf[c->F_cur], c->Fbuf[c->F_cur ^ 1], c->dt, c->cell, c->yee_tile, c->yee_index64, c->yee_wide, st, &c->launches);
    if (e != cudaSuccess) return e;
    c->F_cur ^= 1;
    c->d.Fpad = c->Fbuf[c->F_cur];
    return cudaSuccess;
}

// One step = [sort of the previous step's result, fused into the step kernel's prologue] + gather, push,
// deposit, in-place write-back + convert J + make room + scatter leavers.  The state is left unsorted
// ("dirty"); whoever needs the sorted arrangement (the next step, a load, a read-back) sorts it.
static int enqueue_steps(pic_ctx* c, int n, cudaStream_t st)
{
    PicDev& d = c->d;
    const size_t ncell = (size_t)d.nx * d.ny * d.nz;
    for (int i = 0; i < n; ++i) {
        if (c->dirty && !c->fuse_sort) {
            int rc = ensure_sorted(c);
            if (rc != PIC_OK) return rc;
        }
        // which variants to launch: a belief from the last synchronisation, with a margin; a supercell that crossed
        // the line since is still stepped correctly, by the variant that takes every supercell
        // (the variant that "takes every supercell" steps one of the other class correctly, only slower: a class is
        // dropped when it holds less than 1/64 of the non-empty supercells — a laser pulse that bunches a few hundred
        // of 200 000 sparse supercells past the line must not switch the whole step to the mixed mode)
        d.class_all = 0;
        if (c->n_dense + c->n_sparse > 0) {
            if ((long long)c->n_dense * 64 <= c->n_sparse) d.class_all = 1;
            else if ((long long)c->n_sparse * 64 <= c->n_dense) d.class_all = 2;
        }
        if (c->force_class >= 0) d.class_all = c->force_class;
        // A step that only launches the sparse variant accumulates J in float (shared tile and global array): its
        // supercells see few same-node collisions, and the 64-bit accumulators cost a memset and a convert pass over
        // 3 x 8 B per CELL — on the 67 M-cell grid of configs[2] 4 GB per step, 17 % of the step (profiles/README.md)
        const bool fix = c->fixed_point && !(c->sparse_float && d.class_all == 1);
        cudaError_t e = fix ? cudaMemsetAsync(d.J64, 0, 3 * ncell * sizeof(long long), st)   // S16
                            : cudaMemsetAsync(d.J, 0, 3 * ncell * sizeof(float), st);
        if (e == cudaSuccess) e = cudaMemsetAsync(d.ctr + CTR_EXCH, 0, sizeof(int), st);
        if (e == cudaSuccess) e = cudaMemsetAsync(d.ctr + CTR_OVF, 0, sizeof(int), st);
        if (e == cudaSuccess && c->cell_kernel == 2) e = cudaMemsetAsync(d.ctr + CTR_WORK, 0, sizeof(int), st);
        cudaEvent_t ev0 = nullptr, ev1 = nullptr;
        if (e == cudaSuccess && c->timing) {
            e = cudaEventCreate(&ev0);
            if (e == cudaSuccess) e = cudaEventCreate(&ev1);
            if (e == cudaSuccess) e = cudaEventRecord(ev0, st);
        }
        // An all-sparse step needs no cell order (one thread per particle): it can run on the unsorted state the last
        // step left — holes of leavers, arrivals appended — instead of re-sorting 100 % of the records when a fraction of
        // a percent moved; a sort every nosort_period steps bounds the holes.
        const bool nosort = c->sparse_nosort && c->dirty && c->fuse_sort && d.class_all == 1 &&
                            c->steps_unsorted < c->nosort_period;
        d.nosort = nosort ? 1 : 0;
        d.fused = c->dirty ? 1 : 0;
        if (nosort) {
            // the pending histogram is not consumed by a sort: clear it and let this step fill it again
            if (e == cudaSuccess) e = pic_launch_zero_ints(c->hist[c->hist_cur], (size_t)d.nsc * 256, st, &c->launches);
            d.cell_hist = c->hist[c->hist_cur];
            d.cell_hist_prev = c->hist[c->hist_cur ^ 1];
            ++c->steps_unsorted;
        } else {
            if (c->dirty) d.cur ^= 1;       // the kernel sorts pool cur^1 into pool cur and steps it there
            d.cell_hist_prev = c->hist[c->hist_cur];        // pending histogram (all zero when the state is sorted)
            c->hist_cur ^= 1;
            d.cell_hist = c->hist[c->hist_cur];             // this step's
            c->steps_unsorted = 0;
        }
        if (!nosort && d.fused && d.class_all != 2) {      // sparse supercells: the stand-alone sort, from the other pool into this one
            PicDev ds = d;
            ds.cur = d.cur ^ 1;
            ds.cell_hist = d.cell_hist_prev;
            ds.sort_filter = d.class_all == 1 ? 0 : 1;
            if (e == cudaSuccess) e = pic_launch_sort(ds, st, &c->launches);
        }
        if (e == cudaSuccess) e = pic_launch_step(d, c->order, c->use_tma && c->tmap_ok, fix, c->tmap[c->F_cur], st, &c->launches, c->cell_kernel,
                                                  c->overlap ? c->aux : PicAux{nullptr, nullptr, nullptr});
        d.fused = 0;
        if (e == cudaSuccess && c->timing) {
            e = cudaEventRecord(ev1, st);
            c->events.push_back(ev0);
            c->events.push_back(ev1);
        }
        if (e == cudaSuccess) e = pic_launch_overflow(d, c->order, fix, st, &c->launches);
        if (e == cudaSuccess && fix) e = pic_launch_convert(d, st, &c->launches);
        if (e == cudaSuccess) e = pic_launch_prepare(d, st, &c->launches);
        if (e == cudaSuccess) e = pic_launch_scatter(d, st, &c->launches);
        d.nosort = 0;
        if (e == cudaSuccess && c->field_update) e = enqueue_field_update(c, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "pic_step: launch");
        c->dirty = true;
    }
    return PIC_OK;
}

int32_t pic_step(pic_ctx* c, int32_t n)
{
    if (!c) return PIC_EINVAL;
    if (n < 0) return fail(c, PIC_EINVAL, "pic_step: n < 0");
    if (!c->have_fields) return fail(c, PIC_ESTATE, "pic_step: pic_set_fields has not been called");
    if (c->n_particles == 0) return fail(c, PIC_ESTATE, "pic_step: no particles loaded");
    int rc = enqueue_steps(c, n, c->stream);
    if (rc == PIC_OK) c->steps += n;
    return rc;
}

int32_t pic_update_fields(pic_ctx* c)
{
    if (!c) return PIC_EINVAL;
    if (!c->have_fields) return fail(c, PIC_ESTATE, "pic_update_fields: pic_set_fields has not been called");
    if (!yee_stable(c)) return fail(c, PIC_EINVAL, "pic_update_fields: dt*sqrt(sum 1/cell^2) >= 1 (3-D Yee CFL limit)");
    cudaError_t e = enqueue_field_update(c, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_update_fields: launch");
    return PIC_OK;
}

int32_t pic_get_fields(pic_ctx* c, float* Ex, float* Ey, float* Ez, float* Bx, float* By, float* Bz)
{
    if (!c) return PIC_EINVAL;
    if (!c->have_fields) return fail(c, PIC_ESTATE, "pic_get_fields: pic_set_fields has not been called");
    FieldPtrs f = {{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr}, {Ex, Ey, Ez, Bx, By, Bz}};
    pic_unpad_fields_kernel<<<6u * (unsigned)((c->d.ny + PIC_PADROWS - 1) / PIC_PADROWS) * (unsigned)c->d.nz, 256, 0, c->stream>>>(c->d, f, c->Fbuf[c->F_cur]);
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_fields: unpad kernel");
    return PIC_OK;
}

int32_t pic_get_current(pic_ctx* c, float* Jx, float* Jy, float* Jz)
{
    if (!c) return PIC_EINVAL;
    float* dst[3] = {Jx, Jy, Jz};
    const size_t ncell = (size_t)c->d.nx * c->d.ny * c->d.nz;
    for (int k = 0; k < 3; ++k) {
        if (!dst[k]) continue;
        cudaError_t e = cudaMemcpyAsync(dst[k], c->d.J + k * ncell, ncell * sizeof(float),
                                        cudaMemcpyDeviceToDevice, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_current: cudaMemcpyAsync");
    }
    return PIC_OK;
}

int32_t pic_set_current(pic_ctx* c, const float* Jx, const float* Jy, const float* Jz)
{
    if (!c) return PIC_EINVAL;
    const float* src[3] = {Jx, Jy, Jz};
    const size_t ncell = (size_t)c->d.nx * c->d.ny * c->d.nz;
    for (int k = 0; k < 3; ++k) {
        if (!src[k]) return fail(c, PIC_EINVAL, "pic_set_current: NULL component");
        cudaError_t e = cudaMemcpyAsync(c->d.J + k * ncell, src[k], ncell * sizeof(float), cudaMemcpyDeviceToDevice, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "pic_set_current: cudaMemcpyAsync");
    }
    return PIC_OK;
}

int32_t pic_get_particles(pic_ctx* c, int64_t capacity, int64_t* n_out, double* x, double* y, double* z,
                          float* ux, float* uy, float* uz, float* w, int32_t* species, uint32_t* id,
                          int32_t* supercell)
{
    if (!c) return PIC_EINVAL;
    if (capacity < 0) return fail(c, PIC_EINVAL, "pic_get_particles: capacity < 0");
    {
        int rc = ensure_sorted(c);
        if (rc != PIC_OK) return rc;
    }
    const PicDev& d = c->d;
    pic_scan_counts_kernel<<<1, 1024, 0, c->stream>>>(d);
    GetArgs a;
    a.x = x; a.y = y; a.z = z; a.ux = ux; a.uy = uy; a.uz = uz; a.w = w;
    a.species = species; a.id = id; a.supercell = supercell; a.capacity = capacity;
    a.cx = c->cell[0]; a.cy = c->cell[1]; a.cz = c->cell[2];
    pic_get_particles_kernel<<<d.nsc, 256, 0, c->stream>>>(d, a);
    c->launches += 2;
    long long total = 0;
    cudaError_t e = cudaMemcpyAsync(&total, d.sc_offset + d.nsc, sizeof(long long), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_particles: cudaMemcpyAsync");
    int rc = check_device(c);   // synchronises
    if (n_out) *n_out = total;
    if (rc != PIC_OK) return rc;
    if (total > capacity) return fail(c, PIC_ENOMEM, "pic_get_particles: capacity smaller than the particle count");
    return PIC_OK;
}

int32_t pic_get_counts(pic_ctx* c, int32_t* per_supercell_count)
{
    if (!c) return PIC_EINVAL;
    if (!per_supercell_count) return fail(c, PIC_EINVAL, "pic_get_counts: NULL");
    {
        int rc = ensure_sorted(c);
        if (rc != PIC_OK) return rc;
    }
    cudaError_t e = cudaMemcpyAsync(per_supercell_count, c->d.sc_count, (size_t)c->d.nsc * sizeof(int),
                                    cudaMemcpyDeviceToDevice, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_counts: cudaMemcpyAsync");
    return PIC_OK;
}

int32_t pic_get_stats(pic_ctx* c, int64_t stats[8])
{
    if (!c) return PIC_EINVAL;
    if (!stats) return fail(c, PIC_EINVAL, "pic_get_stats: NULL");
    int ctr[CTR_N];
    unsigned long long c64[CTR64_N];
    cudaError_t e = cudaMemcpyAsync(ctr, c->d.ctr, sizeof ctr, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c64, c->d.ctr64, sizeof c64, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_stats");
    stats[0] = c->n_particles;
    stats[1] = ctr[CTR_LEAVERS_LAST];
    stats[2] = ctr[CTR_POOL_TOP];
    stats[3] = c->d.n_frames;
    stats[4] = ctr[CTR_MAX_COUNT];
    stats[5] = c->steps;
    stats[6] = (int64_t)c64[CTR64_LEAVERS_CUM];
    stats[7] = ctr[CTR_ERROR];
    if (ctr[CTR_ERROR]) return fail(c, PIC_EDEVICE, "pic_get_stats: sticky device fault, see stats[7]");
    return PIC_OK;
}

int32_t pic_sync(pic_ctx* c)
{
    if (!c) return PIC_EINVAL;
    return check_device(c);
}

int32_t pic_set_option(pic_ctx* c, const char* key, int64_t value)
{
    if (!c || !key) return PIC_EINVAL;
    if (!strcmp(key, "tma")) { c->use_tma = value != 0; return PIC_OK; }
    if (!strcmp(key, "class_all")) {
        if (value < -1 || value > 2) return fail(c, PIC_EINVAL, "pic_set_option: class_all must be in -1..2");
        c->force_class = (int)value;
        return PIC_OK;
    }
    if (!strcmp(key, "fuse_sort")) { c->fuse_sort = value != 0; return PIC_OK; }
    if (!strcmp(key, "direct_below")) {
        if (value < 1 || value > (1 << 20)) return fail(c, PIC_EINVAL, "pic_set_option: direct_below out of range");
        if (c->n_particles > 0) return fail(c, PIC_ESTATE, "pic_set_option: set direct_below before loading particles");
        c->d.direct_below = (int)value;
        return PIC_OK;
    }
    if (!strcmp(key, "gather")) {
        // 1 = energy-conserving (Galerkin) gather: implemented in the kernels that gather per particle from the shared
        // tile, so the dense supercells take the one-phase variant of pic_step.cu
        if (value != 0 && value != 1) return fail(c, PIC_EINVAL, "pic_set_option: gather must be 0 or 1");
        if (c->n_particles > 0) return fail(c, PIC_ESTATE, "pic_set_option: set gather before loading particles");
        c->d.gather_ec = (int)value;
        if (value) { c->d.two_phase = 0; c->cell_kernel = 0; }
        return PIC_OK;
    }
    if (!strcmp(key, "sparse_float_tile")) { c->d.sparse_float_tile = value != 0; return PIC_OK; }
    if (!strcmp(key, "sparse_float")) { c->sparse_float = value != 0; return PIC_OK; }
    if (!strcmp(key, "sparse_nosort")) {
        if (value < 0) return fail(c, PIC_EINVAL, "pic_set_option: sparse_nosort must be >= 0");
        c->sparse_nosort = value != 0;
        c->nosort_period = value >= 2 ? (int)(value > 1024 ? 1024 : value) : PIC_NOSORT_PERIOD;
        return PIC_OK;
    }
    if (!strcmp(key, "crowd_first")) { c->d.crowd_min = value ? c->crowd_min_on : (1 << 30); return PIC_OK; }
    if (!strcmp(key, "cell_kernel")) {
        if (value < 0 || value > 2) return fail(c, PIC_EINVAL, "pic_set_option: cell_kernel must be 0, 1 or 2");
        if (value != 0 && c->d.gather_ec) return fail(c, PIC_EINVAL, "pic_set_option: gather = 1 needs cell_kernel = 0");
        c->cell_kernel = (int)value;
        return PIC_OK;
    }
    if (!strcmp(key, "field_update")) {
        if (value != 0 && !yee_stable(c)) return fail(c, PIC_EINVAL, "pic_set_option: field_update needs dt*sqrt(sum 1/cell^2) < 1 (3-D Yee CFL limit)");
        c->field_update = value != 0;
        return PIC_OK;
    }
    if (!strcmp(key, "yee_index64")) { c->yee_index64 = value != 0; return PIC_OK; }
    if (!strcmp(key, "yee_wide")) { c->yee_wide = value != 0; return PIC_OK; }
    if (!strcmp(key, "overlap")) { c->overlap = value != 0; return PIC_OK; }
    if (!strcmp(key, "rest_skip")) { c->d.rest_skip = value != 0; return PIC_OK; }
    if (!strcmp(key, "yee_tile")) {
        if (value != 0 && value != 8 && value != 16) return fail(c, PIC_EINVAL, "pic_set_option: yee_tile must be 0, 8 or 16");
        c->yee_tile = (int)value;
        return PIC_OK;
    }
    if (!strcmp(key, "two_phase") || !strcmp(key, "segment")) {
        // the sorts publish the work-item layout from these two
        if (c->n_particles > 0) return fail(c, PIC_ESTATE, "pic_set_option: set two_phase / segment before loading particles");
        if (key[0] == 't') {
            if (value != 0 && c->d.gather_ec) return fail(c, PIC_EINVAL, "pic_set_option: gather = 1 needs two_phase = 0");
            c->d.two_phase = value != 0;
            return PIC_OK;
        }
        if (value < 2 || value > 16) return fail(c, PIC_EINVAL, "pic_set_option: segment must be in 2..16");
        c->d.seg_num = (int)value;
        return PIC_OK;
    }
    // fault injection (tests): shrink a pool below what pic_workspace_bytes() sized it for, before any particle is
    // loaded; the library must then raise the sticky device error instead of writing out of bounds
    if (!strcmp(key, "limit_frames") || !strcmp(key, "limit_exchange") || !strcmp(key, "limit_tables")) {
        if (c->n_particles > 0) return fail(c, PIC_ESTATE, "pic_set_option: set the limit_* options before loading particles");
        if (value < 0) return fail(c, PIC_EINVAL, "pic_set_option: limit must be >= 0");
        if (key[6] == 'f') c->d.n_frames = (int)(value < c->d.n_frames ? value : c->d.n_frames);
        else if (key[6] == 'e') { c->d.x_cap = (int)(value < c->d.x_cap ? value : c->d.x_cap); }
        else c->d.tbl_pool_size = (int)(value < c->d.tbl_pool_size ? value : c->d.tbl_pool_size);
        return PIC_OK;
    }
    if (!strcmp(key, "deposit")) { c->fixed_point = value != 0; return PIC_OK; }
    if (!strcmp(key, "timing")) { c->timing = value != 0; return PIC_OK; }
    return fail(c, PIC_EINVAL, std::string("pic_set_option: unknown key ") + key);
}

int32_t pic_get_timing(pic_ctx* c, double* step_kernel_ms, int64_t* step_kernel_launches)
{
    if (!c) return PIC_EINVAL;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_timing: synchronize");
    double total = 0.0;
    for (size_t i = 0; i + 1 < c->events.size(); i += 2) {
        float ms = 0.f;
        e = cudaEventElapsedTime(&ms, c->events[i], c->events[i + 1]);
        if (e != cudaSuccess) return cuda_fail(c, e, "pic_get_timing: cudaEventElapsedTime");
        total += ms;
    }
    if (step_kernel_ms) *step_kernel_ms = total;
    if (step_kernel_launches) *step_kernel_launches = (int64_t)(c->events.size() / 2);
    for (cudaEvent_t ev : c->events) cudaEventDestroy(ev);
    c->events.clear();
    return PIC_OK;
}

int64_t pic_launch_count(const pic_ctx* c) { return c ? c->launches : 0; }

const char* pic_last_error(const pic_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int32_t pic_destroy(pic_ctx* c)
{
    if (!c) return PIC_EINVAL;
    for (cudaEvent_t ev : c->events) cudaEventDestroy(ev);
    if (c->aux.fork) cudaEventDestroy(c->aux.fork);
    if (c->aux.join) cudaEventDestroy(c->aux.join);
    if (c->aux.stream) cudaStreamDestroy(c->aux.stream);
    delete c;
    return PIC_OK;
}

}  // extern "C"
