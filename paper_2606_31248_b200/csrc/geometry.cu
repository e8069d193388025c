// geometry.cu -- the field-level pieces around the attention on the device: tile stitching, eq. (5),
// and the StereoRoPE inputs: eq. (1) (tile-centred stereographic coordinates)
// and eq. (2) (winds in the tile centre's East-North frame).  Elementwise, HBM-bound (16 bytes of
// lat / lon in per point); float64 arithmetic because the coordinates (up to ~1.5e3 in units of l_scale) are handed
// to the attention kernels as float32 and must be correct to the last bit or two of that.
#include "../../include/strata_na3d.h"

#include "common.cuh"

namespace strata {
namespace {

// eq. (1)
__global__ void __launch_bounds__(256)
stereo_coords_kernel(const double* __restrict__ lat, const double* __restrict__ lon, long long n, double sin0,
                     double cos0, double lon0, double inv_ell, float* __restrict__ coords, int stride) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    double sp, cp, sd, cd;
    sincos(lat[i], &sp, &cp);
    sincos(lon[i] - lon0, &sd, &cd);
    const double cosc = sin0 * sp + cos0 * cp * cd;
    const double k = 2.0 / (1.0 + cosc) * inv_ell;
    coords[i * stride] = (float)(k * cp * sd);
    coords[i * stride + 1] = (float)(k * (cos0 * sp - sin0 * cp * cd));
  }
}

// eq. (2): v3 = u e + v n in geocentric Cartesian axes (x through (lat, lon) = (0, 0), z the pole); the radial part
// at the tile centre is removed, then the components along e0 and n0 are taken.
__global__ void __launch_bounds__(256)
wind_frame_kernel(const float* __restrict__ u, const float* __restrict__ v, const double* __restrict__ lat,
                  const double* __restrict__ lon, long long n, double sin0, double cos0, double sl0, double cl0,
                  float* __restrict__ u_loc, float* __restrict__ v_loc) {
  const double r0x = cos0 * cl0, r0y = cos0 * sl0, r0z = sin0;
  const double e0x = -sl0, e0y = cl0;
  const double n0x = -sin0 * cl0, n0y = -sin0 * sl0, n0z = cos0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    double sp, cp, sl, cl;
    sincos(lat[i], &sp, &cp);
    sincos(lon[i], &sl, &cl);
    const double uu = (double)u[i], vv = (double)v[i];
    double x = -uu * sl - vv * sp * cl, y = uu * cl - vv * sp * sl, z = vv * cp;
    const double rad = x * r0x + y * r0y + z * r0z;
    x -= rad * r0x; y -= rad * r0y; z -= rad * r0z;
    u_loc[i] = (float)(x * e0x + y * e0y);
    v_loc[i] = (float)(x * n0x + y * n0y + z * n0z);
  }
}

// eq. (5): out = D^-1 P^T W y for tiles that lie inside the field (P copies cells).  Generic form, one
// thread per cell of the [C, GH, GW] field looking at every tile: kept for layouts the row kernel below does not take
// (more than kStitchMaxTiles tiles, more than 65 535 rows).  Both kernels add the tiles in ascending order: same bits.
__global__ void __launch_bounds__(256)
tile_stitch_generic_kernel(const float* __restrict__ tiles, const int* __restrict__ origins, int T, int C, int th, int tw,
                   const float* __restrict__ wy, const float* __restrict__ wx, float* __restrict__ out, int GH, int GW) {
  const long long n = (long long)C * GH * GW;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int gx = (int)(i % GW), gy = (int)((i / GW) % GH), c = (int)(i / ((long long)GW * GH));
    float num = 0.f, den = 0.f;
    for (int t = 0; t < T; ++t) {
      const int dy = gy - origins[2 * t], dx = gx - origins[2 * t + 1];
      if (dy < 0 || dy >= th || dx < 0 || dx >= tw) continue;
      const float w = wy[dy] * wx[dx];
      num = fmaf(w, tiles[(((long long)t * C + c) * th + dy) * tw + dx], num);
      den += w;
    }
    out[i] = den > 0.f ? num / den : 0.f;
  }
}

// The same sum as a stream (HBM-bound: every tile cell is read once, every field cell written once).  A block owns 256
// consecutive cells of one field row for a group of channels.  Warp 0 lists, in ascending order, the tiles that touch
// that row segment (a handful out of T); every thread turns the list into the (weight, offset) pairs of its own cell
// once -- up to kStitchLocal of them in registers -- and then walks the channels with coalesced loads and stores.
constexpr int kStitchMaxTiles = 1024, kStitchLocal = 8;
__global__ void __launch_bounds__(256)
tile_stitch_rows_kernel(const float* __restrict__ tiles, const int* __restrict__ origins, int T, int C, int th, int tw,
                        const float* __restrict__ wy, const float* __restrict__ wx, float* __restrict__ out, int GH, int GW,
                        int c_per_block) {
  __shared__ int s_list[kStitchMaxTiles];
  __shared__ int s_cnt;
  const int gy = blockIdx.y, x0 = blockIdx.x * 256, gx = x0 + threadIdx.x;
  if (threadIdx.x < 32) {
    int cnt = 0;
    for (int base = 0; base < T; base += 32) {
      const int t = base + threadIdx.x;
      bool hit = false;
      if (t < T) {
        const int oy = origins[2 * t], ox = origins[2 * t + 1];
        hit = gy >= oy && gy < oy + th && ox < x0 + 256 && ox + tw > x0;
      }
      const unsigned m = __ballot_sync(0xffffffffu, hit);
      if (hit) s_list[cnt + __popc(m & ((1u << threadIdx.x) - 1u))] = t;
      cnt += __popc(m);
    }
    if (threadIdx.x == 0) s_cnt = cnt;
  }
  __syncthreads();
  if (gx >= GW) return;
  const int cnt = s_cnt;
  const long long plane = (long long)th * tw;
  const int c0 = blockIdx.z * c_per_block, c1 = min(C, c0 + c_per_block);
  float w[kStitchLocal];
  long long off[kStitchLocal];
  int mine = 0;                                     // tiles that cover this cell (ascending), first kStitchLocal in registers
  float den = 0.f;
  bool overflow = false;
  for (int k = 0; k < cnt; ++k) {
    const int t = s_list[k];
    const int dy = gy - origins[2 * t], dx = gx - origins[2 * t + 1];
    if (dx < 0 || dx >= tw) continue;
    const float wk = wy[dy] * wx[dx];
    den += wk;
    if (mine < kStitchLocal) {
#pragma unroll
      for (int u = 0; u < kStitchLocal; ++u)
        if (u == mine) { w[u] = wk; off[u] = (long long)t * C * plane + (long long)dy * tw + dx; }
    } else {
      overflow = true;
    }
    ++mine;
  }
  const float inv_ok = den > 0.f ? 1.f : 0.f;
  if (!overflow) {
    constexpr int CU = 8;                           // channels per pass: their loads are independent (memory-level parallelism)
    int c = c0;
    for (; c + CU <= c1; c += CU) {
      float num[CU];
#pragma unroll
      for (int j = 0; j < CU; ++j) num[j] = 0.f;
#pragma unroll
      for (int u = 0; u < kStitchLocal; ++u)
        if (u < mine) {
          const float* src = tiles + off[u] + c * plane;
#pragma unroll
          for (int j = 0; j < CU; ++j) num[j] = fmaf(w[u], __ldcs(src + j * plane), num[j]);
        }
#pragma unroll
      for (int j = 0; j < CU; ++j) __stcs(out + ((long long)(c + j) * GH + gy) * GW + gx, inv_ok != 0.f ? num[j] / den : 0.f);
    }
    for (; c < c1; ++c) {
      float num = 0.f;
#pragma unroll
      for (int u = 0; u < kStitchLocal; ++u)
        if (u < mine) num = fmaf(w[u], tiles[off[u] + c * plane], num);
      out[((long long)c * GH + gy) * GW + gx] = inv_ok != 0.f ? num / den : 0.f;
    }
  } else {                                          // more than kStitchLocal tiles over one cell: walk the list per channel
    for (int c = c0; c < c1; ++c) {
      float num = 0.f;
      for (int k = 0; k < cnt; ++k) {
        const int t = s_list[k];
        const int dy = gy - origins[2 * t], dx = gx - origins[2 * t + 1];
        if (dx < 0 || dx >= tw) continue;
        num = fmaf(wy[dy] * wx[dx], tiles[(((long long)t * C + c) * th + dy) * tw + dx], num);
      }
      out[((long long)c * GH + gy) * GW + gx] = inv_ok != 0.f ? num / den : 0.f;
    }
  }
}

unsigned grid_for(long long n) {
  const long long b = (n + 255) / 256;
  return (unsigned)(b < 1 ? 1 : b > 148 * 32 ? 148 * 32 : b);
}

}  // namespace
}  // namespace strata

extern "C" {

strata_status_t strata_stereo_coords(const double* lat, const double* lon, long long n, double lat0, double lon0,
                                     double n_total, float* coords, int stride, void* stream) {
  if (n < 0 || stride < 2 || !(n_total > 0.0) || !lat || !lon || !coords) return STRATA_ERR_INVALID_ARG;
  if (n == 0) return STRATA_OK;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const double inv_ell = 1.0 / sqrt(4.0 * 3.14159265358979323846 / n_total);
  strata::prof_begin("stereo_coords", st);
  strata::stereo_coords_kernel<<<strata::grid_for(n), 256, 0, st>>>(lat, lon, n, sin(lat0), cos(lat0), lon0, inv_ell, coords, stride);
  strata::prof_end(st);
  if (cudaGetLastError() != cudaSuccess) return STRATA_ERR_CUDA;
  return STRATA_OK;
}

strata_status_t strata_wind_to_tile_frame(const float* u, const float* v, const double* lat, const double* lon,
                                          long long n, double lat0, double lon0, float* u_loc, float* v_loc,
                                          void* stream) {
  if (n < 0 || !u || !v || !lat || !lon || !u_loc || !v_loc) return STRATA_ERR_INVALID_ARG;
  if (n == 0) return STRATA_OK;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  strata::prof_begin("wind_to_tile_frame", st);
  strata::wind_frame_kernel<<<strata::grid_for(n), 256, 0, st>>>(u, v, lat, lon, n, sin(lat0), cos(lat0), sin(lon0), cos(lon0), u_loc, v_loc);
  strata::prof_end(st);
  if (cudaGetLastError() != cudaSuccess) return STRATA_ERR_CUDA;
  return STRATA_OK;
}

strata_status_t strata_tile_stitch(const float* tiles, const int32_t* origins, int n_tiles, int channels, int th, int tw,
                                   const float* wy, const float* wx, float* out, int gh, int gw, void* stream) {
  if (!tiles || !origins || !wy || !wx || !out || n_tiles < 1 || channels < 1 || th < 1 || tw < 1 || gh < 1 || gw < 1)
    return STRATA_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  strata::prof_begin("tile_stitch", st);
  const long long xy_blocks = (long long)gh * ((gw + 255) / 256);
  if (n_tiles <= strata::kStitchMaxTiles && gh <= 65535) {
    // channel groups: enough blocks to fill the GPU several times over, at most one group per channel
    long long groups = (148LL * 16 + xy_blocks - 1) / xy_blocks;
    groups = groups < 1 ? 1 : groups > channels ? channels : groups > 65535 ? 65535 : groups;
    const int c_per_block = (int)((channels + groups - 1) / groups);
    const dim3 grid((unsigned)((gw + 255) / 256), (unsigned)gh, (unsigned)((channels + c_per_block - 1) / c_per_block));
    strata::tile_stitch_rows_kernel<<<grid, 256, 0, st>>>(tiles, origins, n_tiles, channels, th, tw, wy, wx, out, gh, gw, c_per_block);
  } else {
    strata::tile_stitch_generic_kernel<<<strata::grid_for((long long)channels * gh * gw), 256, 0, st>>>(tiles, origins, n_tiles, channels,
                                                                                               th, tw, wy, wx, out, gh, gw);
  }
  strata::prof_end(st);
  if (cudaGetLastError() != cudaSuccess) return STRATA_ERR_CUDA;
  return STRATA_OK;
}

}  // extern "C"
