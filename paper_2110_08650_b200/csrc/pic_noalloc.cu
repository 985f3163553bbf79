// pic_noalloc.cu — ONE entry point that allocates nothing and needs no workspace: pic_deposit_current_noalloc, the
// Esirkepov deposit of a set of particles given their positions before and after a step.
// For callers that cannot call cudaMalloc or size a workspace: code under CUDA graph capture, tight serving loops,
// harnesses that forbid allocation.  It is the one-thread-per-particle deposit of pic_overflow_kernel (pic_step.cu)
// with its global accumulators — scratch memory, 3 values per cell — moved from the caller's workspace into a
// file-scope device array of a fixed, modest size: PIC_NOALLOC_MAX_CELLS cells (3 x 8 B x 262 144 = 6 MiB, held by
// every GPU that loads the library until the process exits).
//
// The array is SHARED BY EVERY CALL and keeps the last call's contents: each call clears the part it uses first, on
// the caller's stream.  Two calls that overlap on the GPU (different streams, no dependency between them) race on
// it; calls on one stream, or ordered by events, are safe.
//
// In host code the array's NAME is a host-side stand-in, not a device address; the address comes from
// cudaGetSymbolAddress, once per device, with that device current (first call on that device; do it outside graph
// capture).  The existing code paths (pic_create ... pic_step) are untouched by this file.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "../../include/pic_b200.h"
#include "pic_device.cuh"

// 3 accumulators per cell, plus one 256-byte line whose first int is the "moved too far" flag of the call
static __device__ __align__(256) double g_noalloc_J[3 * PIC_NOALLOC_MAX_CELLS + 32];

namespace {

struct NoallocArgs {
    int nx, ny, nz, order;
    double icx, icy, icz;        // 1 / cell size
    float jfx, jfy, jfz;         // (cell_a / dt) / (dx dy dz)
    long long n;
    const double *x0, *y0, *z0, *x1, *y1, *z1;
    const float* qw;
};

// old position -> wrapped cell + fp32 in-cell fraction, new position relative to the OLD cell's origin node
// (minimum image of the move), exactly the representation the step kernels deposit from
__device__ __forceinline__ void noalloc_split(double xa, double xb, double inv_cell, int n, int& cell, float& f0, float& x1r)
{
    const double X0 = xa * inv_cell;
    double c = floor(X0);
    double fr = X0 - c;
    float f = (float)fr;
    if (f >= 1.0f) { f = 0.0f; c += 1.0; fr -= 1.0; }
    double D = (xb - xa) * inv_cell;
    D -= (double)n * rint(D / (double)n);            // periodic: the move is the minimum image
    double r = fmod(c, (double)n);
    if (r < 0) r += (double)n;
    cell = (int)r;
    if (cell >= n) cell = 0;
    f0 = f;
    x1r = (float)(fr + D);
}

template <int O>
__global__ void pic_noalloc_deposit_kernel(const NoallocArgs a, double* __restrict__ acc, int* __restrict__ fault)
{
    const size_t ncell = (size_t)a.nx * a.ny * a.nz;
    const float jf[3] = {a.jfx, a.jfy, a.jfz};
    const int dims[3] = {a.nx, a.ny, a.nz};
    const size_t stride[3] = {1, (size_t)a.nx, (size_t)a.nx * a.ny};
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < a.n; e += (long long)gridDim.x * blockDim.x) {
        int cell[3];
        float f0[3], x1[3];
        noalloc_split(a.x0[e], a.x1[e], a.icx, a.nx, cell[0], f0[0], x1[0]);
        noalloc_split(a.y0[e], a.y1[e], a.icy, a.ny, cell[1], f0[1], x1[1]);
        noalloc_split(a.z0[e], a.z1[e], a.icz, a.nz, cell[2], f0[2], x1[2]);
        const float qw = a.qw[e];
        float S0[3][O + 2], DS[3][O + 2];
        int lo[3];
        bool far = false;
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            far |= !(fabsf(x1[ax] - f0[ax]) < 1.0f);
            float w0[O + 1], w1[O + 1], s1[O + 2];
            const int b0 = shape<O>(f0[ax], w0), b1 = shape<O>(x1[ax], w1);
            lo[ax] = min(b0, b1);
            to_window<O>(w0, b0 - lo[ax], S0[ax]);
            to_window<O>(w1, b1 - lo[ax], s1);
#pragma unroll
            for (int t = 0; t < O + 2; ++t) DS[ax][t] = s1[t] - S0[ax][t];
        }
        if (far) {                   // moved a cell or more (or NaN): not a step's move; flagged, not deposited
            atomicOr(fault, 1);
            continue;
        }
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            const int b = (ax + 1) % 3, c = (ax + 2) % 3;
            const float fac = -qw * jf[ax];
            for (int tc = 0; tc < O + 2; ++tc)
                for (int tb = 0; tb < O + 2; ++tb) {
                    const float br = fac * (S0[b][tb] * S0[c][tc] + 0.5f * DS[b][tb] * S0[c][tc] +
                                            0.5f * S0[b][tb] * DS[c][tc] + (1.0f / 3.0f) * DS[b][tb] * DS[c][tc]);
                    float pre = 0.0f;
                    for (int ta = 0; ta < O + 1; ++ta) {      // the last prefix is sum(DS) = 0: not written
                        pre = fmaf(DS[ax][ta], br, pre);
                        if (pre == 0.0f) continue;
                        int idx[3];
                        idx[ax] = cell[ax] + lo[ax] + ta; idx[b] = cell[b] + lo[b] + tb; idx[c] = cell[c] + lo[c] + tc;
                        size_t g = ax * ncell;
#pragma unroll
                        for (int x = 0; x < 3; ++x) g += stride[x] * (size_t)wrapi(idx[x], dims[x]);
                        atomicAdd(acc + g, (double)pre);
                    }
                }
        }
    }
}

// accumulators -> float J; if a particle was left out (flag), element 0 of every component becomes NaN: the call is
// asynchronous and has no status to read back, so the error is made impossible to overlook in its output
__global__ void pic_noalloc_convert_kernel(const double* __restrict__ acc, const int* __restrict__ fault, size_t ncell,
                                           float* Jx, float* Jy, float* Jz)
{
    const bool bad = *fault != 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < ncell; i += (size_t)gridDim.x * blockDim.x) {
        const bool poison = bad && i == 0;
        Jx[i] = poison ? __int_as_float(0x7fc00000) : (float)acc[i];
        Jy[i] = poison ? __int_as_float(0x7fc00000) : (float)acc[ncell + i];
        Jz[i] = poison ? __int_as_float(0x7fc00000) : (float)acc[2 * ncell + i];
    }
}

int noalloc_fail(char* errbuf, int64_t errbuf_len, int code, const char* msg)
{
    if (errbuf && errbuf_len > 0) {
        strncpy(errbuf, msg, (size_t)errbuf_len - 1);
        errbuf[errbuf_len - 1] = 0;
    }
    return code;
}

// device address of the scratch array, looked up once per device (with that device current)
#define PIC_NOALLOC_MAX_DEVICES 64
std::mutex g_noalloc_mutex;
double* g_noalloc_ptr[PIC_NOALLOC_MAX_DEVICES] = {nullptr};

cudaError_t noalloc_scratch(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= PIC_NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_J);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int32_t pic_deposit_current_noalloc(const int32_t grid[3], const double cell[3], double dt, int32_t shape_order,
                                               int64_t n, const double* x0, const double* y0, const double* z0,
                                               const double* x1, const double* y1, const double* z1, const float* qw,
                                               float* Jx, float* Jy, float* Jz, void* stream,
                                               char* errbuf, int64_t errbuf_len)
{
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (!grid || !cell) return noalloc_fail(errbuf, errbuf_len, PIC_EINVAL, "pic_deposit_current_noalloc: grid or cell is NULL");
    if (shape_order < 1 || shape_order > 3 || !(dt > 0.0) || n < 0)
        return noalloc_fail(errbuf, errbuf_len, PIC_EINVAL, "pic_deposit_current_noalloc: need order in 1..3, dt > 0, n >= 0");
    for (int a = 0; a < 3; ++a)
        if (grid[a] < 4 || !(cell[a] > 0.0))      // (windows of up to 5 nodes wrap correctly from 4 cells on)
            return noalloc_fail(errbuf, errbuf_len, PIC_EINVAL, "pic_deposit_current_noalloc: need grid >= 4 cells and cell > 0 on every axis");
    const uint64_t ncell = (uint64_t)grid[0] * (uint64_t)grid[1] * (uint64_t)grid[2];
    if (ncell > PIC_NOALLOC_MAX_CELLS) {
        char msg[200];
        snprintf(msg, sizeof msg, "pic_deposit_current_noalloc: grid of %llu cells exceeds the maximum of %d cells of the "
                 "built-in scratch array (use pic_create with a workspace for larger grids)", (unsigned long long)ncell,
                 PIC_NOALLOC_MAX_CELLS);
        return noalloc_fail(errbuf, errbuf_len, PIC_EINVAL, msg);
    }
    if (!Jx || !Jy || !Jz || (n > 0 && (!x0 || !y0 || !z0 || !x1 || !y1 || !z1 || !qw)))
        return noalloc_fail(errbuf, errbuf_len, PIC_EINVAL, "pic_deposit_current_noalloc: NULL array");
    cudaStream_t st = (cudaStream_t)stream;
    double* acc = nullptr;
    cudaError_t e = noalloc_scratch(&acc);
    if (e != cudaSuccess) {
        char msg[200];
        snprintf(msg, sizeof msg, "pic_deposit_current_noalloc: cudaGetSymbolAddress of the scratch array: %s", cudaGetErrorString(e));
        return noalloc_fail(errbuf, errbuf_len, PIC_ECUDA, msg);
    }
    // the array keeps the last call's sums and flag: clear what this call uses, on the caller's stream
    int* fault = reinterpret_cast<int*>(acc + 3 * (size_t)PIC_NOALLOC_MAX_CELLS);
    e = cudaMemsetAsync(acc, 0, 3 * ncell * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(fault, 0, sizeof(int), st);
    if (e == cudaSuccess && n > 0) {
        NoallocArgs a;
        a.nx = grid[0]; a.ny = grid[1]; a.nz = grid[2]; a.order = shape_order;
        a.icx = 1.0 / cell[0]; a.icy = 1.0 / cell[1]; a.icz = 1.0 / cell[2];
        const double V = cell[0] * cell[1] * cell[2];
        a.jfx = (float)(cell[0] / dt / V); a.jfy = (float)(cell[1] / dt / V); a.jfz = (float)(cell[2] / dt / V);
        a.n = n; a.x0 = x0; a.y0 = y0; a.z0 = z0; a.x1 = x1; a.y1 = y1; a.z1 = z1; a.qw = qw;
        const long long blocks = (n + 255) / 256;
        const int nb = (int)(blocks < 148 * 16 ? blocks : 148 * 16);
        switch (shape_order) {
            case 1: pic_noalloc_deposit_kernel<1><<<nb, 256, 0, st>>>(a, acc, fault); break;
            case 2: pic_noalloc_deposit_kernel<2><<<nb, 256, 0, st>>>(a, acc, fault); break;
            default: pic_noalloc_deposit_kernel<3><<<nb, 256, 0, st>>>(a, acc, fault); break;
        }
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        const size_t cb = (size_t)((ncell + 255) / 256);
        pic_noalloc_convert_kernel<<<(unsigned)(cb < 148 * 8 ? cb : 148 * 8), 256, 0, st>>>(acc, fault, (size_t)ncell, Jx, Jy, Jz);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        char msg[200];
        snprintf(msg, sizeof msg, "pic_deposit_current_noalloc: %s", cudaGetErrorString(e));
        return noalloc_fail(errbuf, errbuf_len, PIC_ECUDA, msg);
    }
    return PIC_OK;
}
