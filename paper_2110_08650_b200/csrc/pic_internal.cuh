// pic_internal.cuh — device-side state layout shared by the translation units of
// libpic_b200.so.  Nothing here is visible through the C ABI (include/pic_b200.h).
//
// Particle storage ("per-supercell ... fixed-sized
// particle vectors"): a pool of FRAMES of PIC_FRAME slots.  A frame belongs to one
// supercell; a supercell's particles occupy slots [0,count) of its frame list, SORTED BY
// CELL (cell_off[s][c] .. cell_off[s][c+1] are the slots of local cell c).  Per slot one
// 32-byte record (one DRAM sector): float4 {fx,fy,fz,w} (in-cell fraction in [0,1), weight)
// and float4 {ux,uy,uz, bits(local cell | species<<16 | flags<<24)}, plus a uint32 id in a
// parallel array.  Two pools (ping-pong): the step kernel updates records in place in pool
// `cur`, the sort kernel writes the re-sorted supercell into the other pool.
// The frame list of supercell s is tbl_pool[tbl_off[s] .. tbl_off[s]+sc_nframes[s]), the same
// frame indices in both pools.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define PIC_FRAME 256            // slots per frame == threads per step CTA
#define PIC_SCX 8
#define PIC_SCY 8
#define PIC_SCZ 4
#define PIC_SC_CELLS (PIC_SCX * PIC_SCY * PIC_SCZ)
#define PIC_NSPECIES 16
#define PIC_TBL_CLASSES 32
#define PIC_TBL_FREE 2048        // free table regions remembered per capacity class
#define PIC_CROWD_MAX 1024       // CTAs in front of the step kernels' grids reserved for crowded supercells
#define PIC_LEFT_FLAG 0x01000000u   // record bits: the particle left this supercell (hole until the sort)

// device counters (int32 each) in PicDev::ctr
enum {
    CTR_POOL_TOP = 0,     // frames handed out so far
    CTR_TBL_TOP = 1,      // frame-table entries handed out so far
    CTR_EXCH = 2,         // leavers in the exchange buffer (this step)
    CTR_ERROR = 3,        // sticky error word (PIC_DEV_* bits)
    CTR_LEAVERS_LAST = 4,
    CTR_MAX_COUNT = 5,
    CTR_WMAX_BITS = 6,
    CTR_OVF = 7,
    CTR_FREE_TOP = 8,     // entries on the stack of returned frames (may dip below 0 while prepare pops)          // entries in the overflow queue of out-of-window particles (this step)
       // bits of max |weight| loaded so far (non-negative floats order like ints)
    CTR_NDENSE = 12,      // non-empty supercells at or above the sparse/dense line after this step (pic_prepare_kernel)
    CTR_NSPARSE = 13,     // non-empty supercells below it
    CTR_CROWD = 11,       // entries in crowd_list (supercells the next step starts first), built by pic_prepare_kernel
    CTR_WORK = 10,        // next supercell of the persistent step kernel (zeroed before every launch)
    CTR_NEGMIN = 9,       // max over non-empty supercells of (2^30 - population) seen by pic_prepare_kernel, i.e. 2^30 - min
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
    float qmax;                  // max |q| over the species slots in use
    int n_species;               // species ids < n_species are valid
    // frames (two pools, see above)
    float4* rec[2];
    uint32_t* pid[2];
    int cur;                     // pool holding the current state
    int two_phase;               // 1: gather per item with the cell's stencil in registers
    int order;                   // shape order (host copy for kernels that are not templated on it)
    int seg_num;                 // work-item length target in quarters of the mean cell population (2..16)
    int n_frames;
    int* free_stack;             // [n_frames] frames returned by shrinking supercells
    int* tbl_pool;
    int tbl_pool_size;
    int* tbl_off;                // [nsc]
    int* tbl_cap;                // [nsc] capacity of the supercell's table region: 0 or a power of two >= 8
    int* tbl_old_off;            // [nsc] region abandoned by the last growth (pushed on tbl_free by pic_scatter_kernel)
    int* tbl_old_cap;            // [nsc] its capacity, 0 = none
    int* tbl_free;               // [PIC_TBL_CLASSES][PIC_TBL_FREE] offsets of free regions by capacity class (log2)
    int* tbl_free_top;           // [PIC_TBL_CLASSES] entries per class (prepare only pops, scatter only pushes)
    int* sc_nframes;             // [nsc]
    int* sc_count;               // [nsc] particles in the supercell
    int* sc_tail;                // [nsc] slots in use incl. holes of leavers and appended arrivals
    int* cell_off;               // [nsc][257] slot ranges of the local cells (sorted arrangement)
    int* cell_hist;              // [nsc][256] particles per NEW local cell (stayers + arrivals), filled by this step
    int* cell_hist_prev;         // the previous step's histogram, consumed (and cleared) by the fused sort: CTAs of one
                                 // launch read it while others already add this step's leavers to cell_hist
    unsigned char* cell_perm;    // [nsc][256] local cells ordered by decreasing work-item length
    unsigned short* cell_kbase;  // [nsc][256] first work item of the cell at that position
    int* sc_incoming;            // [nsc] leavers headed here
    int* sc_left;                // [nsc] leavers of the last step (written by the step kernel, consumed by prepare)
    int* sc_next;                // [nsc] population after the pending sort (stayers + arrivals), set by prepare
    int* crowd_list;             // [PIC_CROWD_MAX] supercells with >= crowd_min particles: the step kernels start them first
    int* sc_crowd;               // [nsc] 1 = listed in crowd_list (its natural CTA exits)
    int crowd_min;
    int sparse_float_tile;       // option "sparse_float_tile": the sparse variant keeps a float J tile (flushed into J64)
    int float_tile_to_j64;       // set by the launcher for that variant
    int nosort;                  // this step runs on the unsorted state of the last one (all-sparse steps, option "sparse_nosort")
    int rest_skip;               // option "rest_skip": sparse variant, warps of particles at rest in a field-free supercell skip the particle
    int gather_ec;               // option "gather" = 1: energy-conserving gather (per-particle gather paths only)
    int direct_below;            // supercells with fewer particles count as sparse (one thread per particle); option "direct_below"
    int class_all;               // host's belief, from counters read at its last synchronisation (performance only, any
                                 // value is correct): 1 = no supercell is dense: the sparse variant takes every supercell;
                                 // 2 = none is sparse: the dense variant takes every supercell; 0 = classify by population
    int sort_filter;             // pic_sort_kernel: 1 = only supercells of the sparse class (sc_next < 6 per cell)
    int fused;                   // 1: pool cur^1 holds the stepped, not yet sorted state; the step kernel sorts its
                                 //    supercell into pool cur first (sparse supercells were sorted by
                                 //    pic_sort_kernel just before), 0: pool cur is sorted
    // exchange buffer for supercell leavers
    float4* x_rec;               // 2 float4 per entry
    uint32_t* x_id;
    int* x_dst;
    int x_cap;
    float4* ovf;                 // overflow queue of out-of-window particles, 2 float4 per entry
    int ovf_cap;
    // counters
    int* ctr;
    unsigned long long* ctr64;
    // grids
    const float* Fpad;           // the fields (Ex,Ey,Ez,Bx,By,Bz), kept padded with periodic halos only — what the TMA
                                 // tile loads read: [6][nz+PZ][ny+PY][nx+PX]; node (i,j,k) at pic_padded_index()
    int pad_lo_x;                // x halo below node 0 in Fpad = the tile's guard width, so that
                                 // every TMA box starts on a 16-byte boundary
    float* J;                    // 3 components x ncell
    long long* J64;              // fixed-point accumulators of the same shape (deposit option 1)
    // scratch
    long long* sc_offset;        // [nsc+1] exclusive scan of sc_count (pic_get_particles)
};

// padding of the field arrays (periodic halos pre-filled)
#define PIC_PAD_LO 2
#define PIC_PAD_X 8              // nx + 8 keeps the row pitch a multiple of 16 bytes
#define PIC_PAD_Y 4
#define PIC_PAD_Z 4

// element of component c at node (i,j,k), 0 <= i < nx etc., in the padded field array
__host__ __device__ __forceinline__ size_t pic_padded_index(const PicDev& d, int c, int i, int j, int k)
{
    const size_t px = d.nx + PIC_PAD_X, py = d.ny + PIC_PAD_Y, pz = d.nz + PIC_PAD_Z;
    return (size_t)(i + d.pad_lo_x) + px * ((size_t)(j + PIC_PAD_LO) + py * ((size_t)(k + PIC_PAD_LO) + pz * c));
}

// Work items of the step kernel: a cell of n particles is cut into ceil(n/T) segments, with T about
// 3/4 of the supercell's mean cell population (measured optimum of balance vs. flushes).
// Two-phase path: an item's positions and gathered fields sit in shared memory, so an item holds at
// most PIC_ITEM_LMAX particles (what fits beside the tiles with two CTAs per SM) and is flushed once.
#define PIC_ITEM_LMAX(O) ((O) == 3 ? 6 : 11)
#define PIC_DIRECT_BELOW 768     // default of PicDev::direct_below: supercells with fewer particles (< 3 per cell) count as sparse
#define PIC_ITEMCAP 1024         // work items per supercell: <= 256 + count/T

// Work-item length target; lmax > 0 caps it where the supercell's item list still fits PIC_ITEMCAP
// (count <= 768*lmax); more crowded supercells keep longer items and take the one-phase path.
__host__ __device__ inline int pic_segment_target(int supercell_count, int seg_num, int lmax)
{
    int t = (seg_num * supercell_count + 1023) / 1024;     // seg_num/4 of the mean cell population
    if (t < 4) t = 4;
    if (t > 256) t = 256;      // PIC_FLUSH_MAX: the fixed-point split of a register sum is exact for <= 256 contributions
    if (lmax > 0 && supercell_count <= 768 * lmax) t = lmax;    // two-phase: items as long as the staging allows
    return t;
}

// Which supercell a step CTA works on: the first PIC_CROWD_MAX CTAs of the grid take the crowded supercells that
// pic_prepare_kernel listed (one CTA walks 100 k particles while ordinary supercells take 4 k: started last, such a
// CTA is the tail of the whole launch; started first, the others fill in around it), the rest their own index.
// Returns -1 for a CTA without work.
__device__ inline int pic_cta_supercell(const PicDev& d, int block)
{
    if (d.crowd_min >= (1 << 30)) return block;      // option crowd_first off (default): the grid has no extra CTAs
    if (block < PIC_CROWD_MAX) return block < d.ctr[CTR_CROWD] ? d.crowd_list[block] : -1;
    const int s = block - PIC_CROWD_MAX;
    return d.sc_crowd[s] ? -1 : s;
}

// CTAs of a step-kernel launch (see pic_cta_supercell)
inline int pic_step_grid(const PicDev& d) { return d.nsc + (d.crowd_min >= (1 << 30) ? 0 : PIC_CROWD_MAX); }

__host__ __device__ inline uint32_t pic_pack_bits(int local_cell, int species)
{
    return (uint32_t)local_cell | ((uint32_t)species << 16);
}

// launchers implemented in pic_step.cu
// aux: a second stream with its fork/join events (or aux.stream == nullptr): the two dense variants, which take disjoint
// supercells, then run side by side — the crowded supercells' few long CTAs first, the ordinary ones filling the SMs
struct PicAux { cudaStream_t stream; cudaEvent_t fork, join; };
cudaError_t pic_launch_step(const PicDev& d, int order, bool use_tma, bool fixed_point, const void* tmap,
                            cudaStream_t st, int64_t* launches, int cell_kernel, const PicAux& aux);
// pic_cell.cu: the dense whole-cell kernel (fixed point), launched over all supercells; sparse ones exit
cudaError_t pic_launch_cell(const PicDev& d, int order, bool use_tma, const void* tmap, cudaStream_t st, int64_t* launches,
                            bool persistent);
cudaError_t pic_launch_overflow(const PicDev& d, int order, bool fixed_point, cudaStream_t st, int64_t* launches);
cudaError_t pic_launch_convert(const PicDev& d, cudaStream_t st, int64_t* launches);
cudaError_t pic_launch_zero_ints(int* p, size_t n, cudaStream_t st, int64_t* launches);   // n a multiple of 4
cudaError_t pic_launch_prepare(const PicDev& d, cudaStream_t st, int64_t* launches);
cudaError_t pic_launch_scatter(const PicDev& d, cudaStream_t st, int64_t* launches);
cudaError_t pic_launch_sort(const PicDev& d, cudaStream_t st, int64_t* launches);   // pool cur -> the other
// pic_fields.cu: one Yee update, padded array F_in (level n) -> padded array F_out (level n+1, all periodic images), J = d.J
cudaError_t pic_launch_yee(const PicDev& d, const float* F_in, float* F_out, double dt, const double cell[3], int tile_y,
                           bool index64, bool wide, cudaStream_t st, int64_t* launches);
