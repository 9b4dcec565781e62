// tmap.h - host-side TMA tensor-map helpers shared by the tcgen05 kernels (internal).
#pragma once
#include <cuda.h>
#include <stdint.h>

#include <string>

namespace pulse {
namespace tmap {

struct Tap { int dx, dy, px, py, widx; };

// bf16 tensor map, 128-byte swizzle; dims/box innermost first; strides (bytes) for dims 1..rank-1.  Cached.
bool get_map(const void* ptr, int rank, const uint64_t* dims, const uint64_t* strides, const uint32_t* box,
             CUtensorMap* out, int swizzle_bytes = 128, int elem_bytes = 2);     // elem_bytes 2: bf16, 4: fp32
// row-major fp32 [rows][cols] matrix with an unswizzled (bcols, brows) box
bool mat_map_f32(const void* ptr, uint64_t rows, uint64_t cols, int bcols, int brows, CUtensorMap* out);
// NHWC activation [n,h,w,c] as a 4-D map (c, w, h, n) with box (64, bw, bh, bn)
bool act_map(const void* ptr, int n, int h, int w, int c, int bw, int bh, int bn, CUtensorMap* out);
// stride-2 parity view (px*c + ch, x', py, y', n) of [n,h,w,c], box (64, bw, 1, bh, bn)
bool act_map_s2(const void* ptr, int n, int h, int w, int c, int bw, int bh, int bn, CUtensorMap* out);
// row-major [rows][k] matrix, box (64, brows)
bool mat_map(const void* ptr, uint64_t rows, uint64_t k, int brows, CUtensorMap* out);
// pixel-grid tiling of 128 pixels: bw = W (W | 128), then rows, then images
bool tile_geometry(int gh, int gw, int& bw, int& bh, int& bn);
bool tile_geometry64(int gh, int gw, int& bw, int& bh, int& bn);
bool act_map_c(const void* ptr, int n, int h, int w, int c, int cbox, int bw, int bh, int bn, CUtensorMap* out);
// the parity view with a (cbox, bw, 1, bh, bn) box; swizzle = 2 * cbox bytes
bool act_map_s2_c(const void* ptr, int n, int h, int w, int c, int cbox, int bw, int bh, int bn, CUtensorMap* out);
int sm_count();
void set_error(const std::string& e);
const std::string& last_error();

}  // namespace tmap
}  // namespace pulse
