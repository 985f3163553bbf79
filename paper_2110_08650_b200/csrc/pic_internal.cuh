// pic_internal.cuh — device-side state layout shared by the translation units of
// libpic_b200.so.  Nothing here is visible through the C ABI (include/pic_b200.h).
//
// Particle storage ("per-supercell ... fixed-sized
// particle vectors"): a pool of FRAMES of PIC_FRAME slots.  A frame belongs to one
// supercell; a supercell's particles occupy slots [0,count) of its frame list, densely.
// Per slot: float4 pos = {fx,fy,fz,w} (in-cell fraction in [0,1), weight),
//           float4 mom = {ux,uy,uz, bits(local cell | species<<16)},
//           uint32  id.
// The frame list of supercell s is tbl_pool[tbl_off[s] .. tbl_off[s]+sc_nframes[s]).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define PIC_FRAME 256            // slots per frame == threads per step CTA
#define PIC_SCX 8
#define PIC_SCY 8
#define PIC_SCZ 4
#define PIC_SC_CELLS (PIC_SCX * PIC_SCY * PIC_SCZ)
#define PIC_NSPECIES 16

// device counters (int32 each) in PicDev::ctr
enum {
    CTR_POOL_TOP = 0,     // frames handed out so far
    CTR_TBL_TOP = 1,      // frame-table entries handed out so far
    CTR_EXCH = 2,         // leavers in the exchange buffer (this step)
    CTR_ERROR = 3,        // sticky error word (PIC_DEV_* bits)
    CTR_LEAVERS_LAST = 4,
    CTR_MAX_COUNT = 5,
    CTR_WMAX_BITS = 6,    // bits of max |weight| loaded so far (non-negative floats order like ints)
    CTR_N = 16
};
// 64-bit counters in PicDev::ctr64
enum { CTR64_LEAVERS_CUM = 0, CTR64_N = 4 };

struct PicDev {
    // geometry
    int nx, ny, nz;
    int nsx, nsy, nsz, nsc;
    float dtdx, dtdy, dtdz;      // dt / cell size: displacement in cells per unit velocity
    float jfx, jfy, jfz;         // (cell_a / dt) / (dx dy dz): J factor without q*w
    float h[PIC_NSPECIES];       // (q/m) dt / 2
    float q[PIC_NSPECIES];
    float qmax;                  // max |q| over the species table
    // frames
    float4* pos;
    float4* mom;
    uint32_t* pid;
    int n_frames;
    int* tbl_pool;
    int tbl_pool_size;
    int* tbl_off;                // [nsc]
    int* tbl_cap;                // [nsc]
    int* sc_nframes;             // [nsc]
    int* sc_count;               // [nsc] particles in the supercell
    int* sc_stay;                // [nsc] stayers after the step kernel's compaction
    int* sc_incoming;            // [nsc] leavers headed here
    // exchange buffer for supercell leavers
    float4* x_pos;
    float4* x_mom;
    uint32_t* x_id;
    int* x_dst;
    int x_cap;
    // counters
    int* ctr;
    unsigned long long* ctr64;
    // grids
    const float* F;              // 6 components x ncell (Ex,Ey,Ez,Bx,By,Bz), unpadded
    const float* Fpad;           // padded copy for TMA: [6][nz+PZ][ny+PY][nx+PX]
    int pad_lo_x;                // x halo below node 0 in Fpad = the tile's guard width, so that
                                 // every TMA box starts on a 16-byte boundary
    float* J;                    // 3 components x ncell
    long long* J64;              // fixed-point accumulators of the same shape (deposit option 1)
    // scratch
    long long* sc_offset;        // [nsc+1] exclusive scan of sc_count (pic_get_particles)
};

// padding of the TMA copy of the fields (periodic halos pre-filled)
#define PIC_PAD_LO 2
#define PIC_PAD_X 8              // nx + 8 keeps the row pitch a multiple of 16 bytes
#define PIC_PAD_Y 4
#define PIC_PAD_Z 4

__host__ __device__ inline uint32_t pic_pack_bits(int local_cell, int species)
{
    return (uint32_t)local_cell | ((uint32_t)species << 16);
}

// launchers implemented in pic_step.cu
cudaError_t pic_launch_step(const PicDev& d, int order, bool use_tma, bool fixed_point, const void* tmap,
                            cudaStream_t st, int64_t* launches);
cudaError_t pic_launch_resort(const PicDev& d, cudaStream_t st, int64_t* launches, bool scatter);
