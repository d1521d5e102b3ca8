// K10: scan -> spherical range image.  "We build each scan as a spherical range image and
// render the Gaussian map under the same spherical projection pi_s"; M_D = [D > 0];
// the image of the tracker's normals N_g-icp.  Readings R25-R27 of DESIGN.md: the grid is the
// renderer's (R1), points are in the sensor frame, the nearest return of a pixel wins (z-buffer), equal fp32 ranges
// break by the lower point index.
// Three kernels, overlapped with programmatic dependent launch (each becomes resident beside its predecessor and waits
// only where it needs its output): clear the z-buffer; one thread per point: pixel from fp64 atan2 (the decision "which pixel" is an
// integer taken in fp64 on both sides of the parity test), 64-bit atomicMin of (range bits << 32 | point index);
// one thread per pixel: range and normal of the winner.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr unsigned long long kEmpty = ~0ull;

struct ScanArgs {
  const float* points; const float* normals;
  long long M;
  int H, W;
  double elev_max, dphi, dth;
  float r_min, r_max;
  unsigned long long* zbuf;
  float* out_range; float* out_normal;
};

__global__ void __launch_bounds__(256) scan_clear_kernel(unsigned long long* zbuf, size_t n) {
  asm volatile("griddepcontrol.launch_dependents;");     // the splat kernel projects its points beside this grid
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) zbuf[k] = kEmpty;
}

// Launched with programmatic stream serialisation beside the clear kernel: the projection of the point (the fp64 part)
// needs nothing from it; griddepcontrol.wait precedes the first touch of the z-buffer and is executed on every path.
__device__ __forceinline__ bool scan_pixel(const ScanArgs& a, long long k, size_t* px, float* r32_out) {
  if (k >= a.M) return false;
  const double x = a.points[3 * k], y = a.points[3 * k + 1], z = a.points[3 * k + 2];
  const double r = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)));
  const float r32 = __double2float_rn(r);
  if (!isfinite(r) || !(r32 > 0.f) || !(r32 >= a.r_min) || !(r32 <= a.r_max)) return false;
  const double phi = atan2(y, x);
  const double th = atan2(z, __dsqrt_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y))));
  const double fc = floor(__ddiv_rn(__dadd_rn(phi, kPi), a.dphi));
  const double fr = floor(__ddiv_rn(__dsub_rn(a.elev_max, th), a.dth));
  if (!isfinite(fc) || !isfinite(fr) || !(fr >= 0.0) || !(fr < (double)a.H)) return false;
  long long col = (long long)fc;
  if (col >= a.W) col -= a.W;                                    // phi = +pi -> column 0
  if (col < 0 || col >= a.W) return false;
  *px = (size_t)fr * a.W + (size_t)col;
  *r32_out = r32;
  return true;
}

__global__ void __launch_bounds__(256) scan_splat_kernel(const ScanArgs a) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  asm volatile("griddepcontrol.launch_dependents;");     // the resolve kernel becomes resident and waits for this grid
  size_t px = 0;
  float r32 = 0.f;
  const bool hit = scan_pixel(a, k, &px, &r32);
  asm volatile("griddepcontrol.wait;" ::: "memory");     // the z-buffer is cleared
  if (hit) atomicMin(&a.zbuf[px], ((unsigned long long)__float_as_uint(r32) << 32) | (unsigned long long)(unsigned int)k);
}

__global__ void __launch_bounds__(256) scan_resolve_kernel(const ScanArgs a) {
  const size_t HW = (size_t)a.H * a.W;
  const size_t px = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  asm volatile("griddepcontrol.wait;" ::: "memory");     // launched beside the splat kernel: wait for its z-buffer
  if (px >= HW) return;
  const unsigned long long e = a.zbuf[px];
  float r = 0.f, nx = 0.f, ny = 0.f, nz = 0.f;
  if (e != kEmpty) {
    r = __uint_as_float((unsigned int)(e >> 32));
    if (a.normals) {
      const size_t k = (size_t)(unsigned int)e;
      nx = a.normals[3 * k]; ny = a.normals[3 * k + 1]; nz = a.normals[3 * k + 2];
    }
  }
  a.out_range[px] = r;
  if (a.out_normal) { a.out_normal[px] = nx; a.out_normal[HW + px] = ny; a.out_normal[2 * HW + px] = nz; }
}

}  // namespace

cudaError_t launch_scan(const SensorDev& sd, const float* points, const float* normals, int64_t M, void* zbuf,
                        float* out_range, float* out_normal, cudaStream_t st) {
  ScanArgs a;
  a.points = points; a.normals = normals; a.M = M;
  a.H = sd.H; a.W = sd.W; a.elev_max = sd.elev_max; a.dphi = sd.dphi; a.dth = sd.dth;
  a.r_min = sd.r_min; a.r_max = sd.r_max;
  a.zbuf = static_cast<unsigned long long*>(zbuf);
  a.out_range = out_range; a.out_normal = out_normal;
  const size_t HW = (size_t)sd.H * sd.W;
  const unsigned gpx = (unsigned)((HW + 255) / 256);
  scan_clear_kernel<<<gpx < (unsigned)sm_count() * 8u ? gpx : (unsigned)sm_count() * 8u, 256, 0, st>>>(a.zbuf, HW);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (M > 0) {
    e = launch_pdl(scan_splat_kernel, dim3((unsigned)((M + 255) / 256)), dim3(256), 0, st, a);
    if (e != cudaSuccess) return e;
  }
  return launch_pdl(scan_resolve_kernel, dim3(gpx), dim3(256), 0, st, a);
}

}  // namespace lgs
