// synim_device.h -- structures shared by the host side of the C ABI (synim_api.cu) and the
// sm_100a kernels (synim_strip.cu, synim_kernels.cu).  Internal; the public interface is include/synim.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace synim {

constexpr int kMaxWfsPerLaunch = 16;   // per-launch WFS batch (kernel-parameter space is 4 KB)
constexpr int kWmapPadRows = 8;        // rows of zeros below each sensor's weight map (the kernel's look-ahead)
constexpr int kSubapGeneral = 1 << 30; // flag in a row-map entry: valid subaperture whose pixel weights differ
constexpr int kSubapRowMask = kSubapGeneral - 1;
constexpr int kStripMaxCols = 30;      // D columns of a strip (one per lane, plus a halo lane on either side)
// edge repair: class of a pixel of the interpolated screen.  Bit 0: the pixel belongs to the strict
// core.  Otherwise bits 1..4 say in which of the directions +x, -x, +y, -y the neighbour P1 is a core pixel (any of
// them set: a ring pixel), bits 5..8 whether the next pixel P2 in that direction is one too.
constexpr int kRepairCore = 1, kRepairP1Shift = 1, kRepairP2Shift = 5, kRepairRingMask = 0x1e;
constexpr int kRepairReach = 2;        // a restored pixel reads up to two pixels away
// tile kernel: per-warp scratch in which the lanes' partial sums of kEdgeBatch edge-sum units wait to be combined:
// per unit 33 floats of column sums, 33 of row-pair differences, 66 of packed interior samples
constexpr int kTileWarpsPerCta = 4, kEdgeBatch = 8, kEdgeSlotFloats = 33 + 33 + 66;
constexpr int kTileScratchBytesPerCta = kTileWarpsPerCta * kEdgeBatch * kEdgeSlotFloats * 4;

// One sensor as the kernel sees it.  All coordinates are ABSOLUTE pixel indices: WFS pixel (i, j)
// (row, column) samples the source grid at
//   col = fwd[0]*j + fwd[1]*i + fwd[2],   row = fwd[3]*j + fwd[4]*i + fwd[5]
// (the centring terms (M-1)/2, (Nx-1)/2, (Ny-1)/2 of synim.h are folded into fwd[2], fwd[5] in
// float64 on the host), and inv is the inverse map  j = inv[0]*col + inv[1]*row + inv[2],
// i = inv[3]*col + inv[4]*row + inv[5].
struct WfsDev {
    double fwd[6];
    double inv[6];
    const float *wmap;       // [M][M]  0.5*P/W_S, 0 where the subaperture is invalid
    const float *gx, *gy;    // [M][M]  G-tilt coefficients (gtilt_maps_kernel); same rows of zeros below
    const int *subap_row;    // [n_subap^2] index among the valid subapertures (| kSubapGeneral if its pixel weights
                             // differ), -1 if invalid
    const unsigned short *rcode;   // edge repair only: [(M+2)][(M+2)] class of every pixel of the halo grid -1..M
                                   // (kRepair* bits below), built per call by repair_maps
    float scale;             // slope_scale
    float w_uniform;         // 0.5 / n_pix^2: the weight of every pixel of a uniform subaperture
    int M, n_subap, n_pix;
    int spb;                 // subapertures per strip when strips are aligned to subaperture columns
                             // (floor(30 / n_pix)); 0: subapertures wider than a strip, unaligned strips
    int red_steps;           // ceil(log2(n_pix)) capped at 5: shuffle steps of the segmented lane reduction
    unsigned npx_magic;      // ceil(2^32 / n_pix): x / n_pix = umulhi(x, npx_magic) for the pixel indices met here
    int row_x, row_y;        // first row of the x / y slopes of this sensor inside a column
    int tab_off, tab_cap;    // this sensor's slice of the CTA's slope table (floats)
    // dense modes, tiles of the WFS grid (synim_tile_kernel): a tile is tile_ns strips x tile_nr subaperture rows
    int tile_ns, tile_nr;    // strips (of spb subapertures) and subaperture rows per tile
    int tiles_x, tiles_y;    // tiles across / down the sensor
    int tile_first;          // index of this sensor's first tile among the launch's tiles of one mode
    int box_pitch, box_h;    // the staged pre-image of a tile: floats per row (multiple of 4), rows
};

struct ImParams {
    const float *cube;       // [n_modes][ny][nx]
    const int *bbox;         // [n_modes][4] or nullptr
    const int *diag;         // [n_modes][4] min/max of x+y, min/max of x-y over the support, or nullptr
    const int *origin;       // [n_modes][2] source pixel of cube pixel (0, 0) of each mode (packed cube), or nullptr
    float *out;              // column-major IM
    long long ld;
    int n_modes, ny, nx, n_wfs;
    int patch_pitch, patch_h;   // the staged box (TMA), floats x rows
    int zero_begin, zero_count; // rows [zero_begin, zero_begin+zero_count) of a column are zeroed by the mode's
                                // CTA (0: the caller cleared them, dense modes)
    int chunks;                 // CTAs per mode (grid.y): the pieces of a dense mode are spread over them
    float patch_pitchf;         // patch_pitch as float (an FFMA operand straight from constant memory)
    unsigned addr_bias;         // (bits of 1.5*2^23) << 2 mod 2^32, see process_strip
    int tab_floats;             // size of the CTA's slope table (multiple of 4)
    int tiles_total;            // tile kernel: tiles of one mode over all sensors of the launch
    int unit_rows;              // 1: aligned sensors' footprints are rounded out to whole subaperture rows (packed zonal walk)
    int reach;                  // extra pixels around a tile / a footprint that a sample may touch: 0, or kRepairReach
    WfsDev wfs[kMaxWfsPerLaunch];
};

// tile kernel: one TMA descriptor per sensor (the boxes differ with the sensors' rotations); 128 bytes each,
// 64-byte aligned as the hardware wants
struct alignas(64) TileMaps {
    unsigned char m[kMaxWfsPerLaunch][128];
};

// launchers; all asynchronous on `stream`, return the launch status.
// The hot path (synim_strip.cu); tensor_map points at a host CUtensorMap over the cube with box
// {patch_pitch, patch_h, 1}
// (p.unit_rows selects the packed zonal walk: numerical derivative, aligned sensors, no repair; the launcher adds the
// warps' scratch to smem_bytes)
cudaError_t launch_strip(const ImParams &p, const void *tensor_map, size_t smem_bytes, bool gtilt, bool repair,
                         cudaStream_t stream);
// Dense modes over sensors whose subapertures fit a strip: one CTA per (mode, sensor, tile of the WFS grid);
// maps.m[w] is sensor w's CUtensorMap over the cube with box {box_pitch, box_h, 1}
cudaError_t launch_tiles(const ImParams &p, const TileMaps &maps, size_t smem_bytes, bool gtilt, bool repair,
                         cudaStream_t stream);
// Edge repair, per call and sensor: the mask [ny][nx] is interpolated through the sensor's map fwd
// (float64), thresholded into the strict core, and turned into (a) the pixel classes rcode [(M+2)^2], (b) the
// reduction weights wmap_out = 0.5*P*core / sum_S(P*core) (from wmap_in = 0.5*P/W_S), (c) the row map rows_out =
// rows_in with kSubapGeneral set unless the subaperture and the pixels its edge sums read are all core.
// core is scratch: (M+2)^2 bytes.
cudaError_t launch_repair_maps(const float *d_mask, int ny, int nx, const double *fwd, double threshold, int n_subap, int n_pix,
                               const float *wmap_in, const int *rows_in, unsigned char *core, unsigned short *rcode,
                               float *wmap_out, int *rows_out, cudaStream_t stream);
cudaError_t launch_subap_weights(const float *d_pupil, const uint8_t *d_valid, int n_subap, int n_pix,
                                 float *d_wmap, int *d_subap_row, int *d_error_flag, cudaStream_t stream);
cudaError_t launch_gtilt_maps(const float *d_pupil, const uint8_t *d_valid, int n_subap, int n_pix, float *d_gx, float *d_gy,
                              cudaStream_t stream);
cudaError_t launch_compute_bboxes(const float *d_cube, int n_modes, int ny, int nx, int *d_bbox, int *d_diag,
                                  cudaStream_t stream);
cudaError_t launch_bbox_extent(const int *d_bbox, int n_modes, int *d_wh, cudaStream_t stream);
size_t max_dynamic_smem();  // opt-in limit of the current device (bytes)
void note_launch();           // every launcher calls this once per kernel it enqueues (synim_launch_count)
long long launches_so_far();

}  // namespace synim
