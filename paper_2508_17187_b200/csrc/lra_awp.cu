// lra_awp.cu -- the data-dependent part of the kernel of Eq. 27 (Table 2) and per-element Mueller
// CFs; SURVEY.md Sec. 8(f) NEXT-3.  Readings R27-R29.
//     c_ij = CF_ij(nu, w, t)  f(ds_i - ds_j)  e^{2 pi i [s_o - (s(P) + ds_i + ds_j)] . u}
// The factor after CF_ij depends on the GRID PIXEL the tap lands on, u_X = (X - nx/2)/scale_u, and on the row's entry
// (f, dl, dm) of a caller-supplied table.  Two ways of applying it, chosen by how many rows share an entry:
//   * every row of the call shares one entry (mosaic imaging: one call per pointing, Table 2 rows 3-4 without PO):
//     G and D run through the tiled region kernels unchanged and the factor is applied to the whole grid once,
//     lra_phase_gradient_kernel -- HBM-bound, 16-24 bytes per pixel and plane;
//   * rows have their own entries (antenna pointing-offset correction, Table 2 "with PO correction"): direct kernels,
//     one CTA (gridding) or warp (degridding) per visibility point, the 2 S phasors of the point's footprint computed
//     in fp64 (sincospi) into shared memory and multiplied into every tap.
// Mueller elements are a loop over elements on a one-plane plan: re-bin with the element's kernel indices, gather the
// element's visibility correlation, grid onto / degrid from the element's grid plane.
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "lra_pipe.cuh"

int lra_sumwt_launch(lra_plan* p, const float* wt, const float* tau, double* sumwt);   // lra_grid.cu

namespace {

__device__ __forceinline__ void lra_awp_red_add(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

// e^{sign 2 pi i turns}, fp64 argument reduction, fp32 result
__device__ __forceinline__ float2 lra_phasor(double turns) {
  double s, c;
  sincospi(2.0 * turns, &s, &c);
  return make_float2((float)c, (float)s);
}

// tab[X] = e^{2 pi i sign a (X - nx/2)} for X < nx;  tab[nx + Y] = f e^{2 pi i sign b (Y - ny/2)} for Y < ny
__global__ void __launch_bounds__(256)
lra_gradient_table_kernel(float2* __restrict__ tab, int nx, int ny, double a, double b, double f) {
  for (int e = blockIdx.x * 256 + threadIdx.x; e < nx + ny; e += gridDim.x * 256) {
    if (e < nx) {
      tab[e] = lra_phasor(a * (double)(e - nx / 2));
    } else {
      const float2 ph = lra_phasor(b * (double)(e - nx - ny / 2));
      tab[e] = make_float2((float)f * ph.x, (float)f * ph.y);
    }
  }
}

// dst (+)= tab[X] * tab[nx + Y] * src for every plane
template <bool ACC>
__global__ void __launch_bounds__(256)
lra_phase_gradient_kernel(const float2* __restrict__ src, const float2* __restrict__ tab, float2* dst, int nx, int ny,
                          long long n) {
  for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n; i += gridDim.x * 256ll) {
    const long long r = i / nx;
    const int X = (int)(i - r * nx), Y = (int)(r % ny);
    const float2 cx = tab[X], ry = tab[nx + Y];
    const float2 ph = make_float2(cx.x * ry.x - cx.y * ry.y, cx.x * ry.y + cx.y * ry.x);
    const float2 v = src[i];
    float2 o = make_float2(v.x * ph.x - v.y * ph.y, v.x * ph.y + v.y * ph.x);
    if (ACC) { const float2 d = dst[i]; o.x += d.x; o.y += d.y; }
    dst[i] = o;
  }
}

struct lra_po_args {
  const double* table;   // device [n_po][3]
  const int32_t* index;  // device [nrow] or null
  int n_po;
  double inv_su, inv_sv; // wavelengths per pixel
};

// phasors of the footprint of one point into shared memory: ph[i] (columns), ph[S + j] (rows, times f); false = skip
__device__ __forceinline__ bool lra_po_phasors(const lra_po_args& po, long long row, int ix, int iy, int S, int nx, int ny,
                                               float2* ph, int t, int nt) {
  const int e = po.index ? po.index[row] : 0;
  if (e < 0 || e >= po.n_po) return false;
  const double f = po.table[3 * e], a = po.table[3 * e + 1] * po.inv_su, b = po.table[3 * e + 2] * po.inv_sv;
  const int h = (S - 1) >> 1;
  for (int q = t; q < 2 * S; q += nt) {
    if (q < S) {
      ph[q] = lra_phasor(a * (double)(ix - h + q - nx / 2));
    } else {
      const float2 r = lra_phasor(b * (double)(iy - h + (q - S) - ny / 2));
      ph[q] = make_float2((float)f * r.x, (float)f * r.y);
    }
  }
  return true;
}

// one CTA walks visibility points; its 256 threads split the S*S taps; every tap update is two red.global.add.f32
__global__ void __launch_bounds__(256)
lra_grid_po_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                   const float* __restrict__ slabs, const float2* __restrict__ vis, const float* __restrict__ wt,
                   const float* __restrict__ tau, int nchan, int ncorr, int nterms, int nx, int ny, int tile_x,
                   lra_po_args po, float2* __restrict__ grid) {
  __shared__ float2 ph[2 * 129];
  const long long n = (long long)counters[0];
  const size_t plane = (size_t)nx * ny;
  for (long long i = blockIdx.x; i < n; i += gridDim.x) {
    const lra_rec r = rec[i];
    const int ix = r.x & 0xffff, iy = r.x >> 16, S = r.w & 0xff, h = (S - 1) >> 1;
    const float2* slab = reinterpret_cast<const float2*>(slabs + ((size_t)r.y << 2));
    const uint32_t k = r.z;
    const int c = (int)(k % (uint32_t)nchan);
    __syncthreads();   // the previous point's phasors are no longer read
    const bool ok = lra_po_phasors(po, (long long)(k / (uint32_t)nchan), ix, iy, S, nx, ny, ph, threadIdx.x, 256);
    __syncthreads();
    if (!ok) continue;   // uniform over the CTA
    float2 val[16];
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        float2 v = make_float2(0.f, 0.f);
        if (t < nterms && p < ncorr) {
          const float w = wt[(size_t)k * ncorr + p] * (tau ? tau[c * nterms + t] : 1.0f);
          const float2 x = vis[(size_t)k * ncorr + p];
          v = make_float2(w * x.x, w * x.y);
        }
        val[t * 4 + p] = v;
      }
    for (int e = threadIdx.x; e < S * S; e += 256) {
      const int j = e / S, ii = e - j * S;
      const float2 c0 = slab[lra_tap_index(S, tile_x, j, ii)];
      const float2 a = ph[ii], b = ph[S + j];
      const float2 f = make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
      const float2 cf = make_float2(c0.x * f.x - c0.y * f.y, c0.x * f.y + c0.y * f.x);
      const size_t pix = (size_t)(iy - h + j) * nx + (ix - h + ii);
#pragma unroll
      for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int p = 0; p < 4; ++p)
          if (t < nterms && p < ncorr) {
            const float2 v = val[t * 4 + p];
            float* g = (float*)(grid + (size_t)(t * ncorr + p) * plane + pix);
            lra_awp_red_add(g, cf.x * v.x - cf.y * v.y);
            lra_awp_red_add(g + 1, cf.x * v.y + cf.y * v.x);
          }
    }
  }
}

// one warp per visibility point
template <int NC>
__global__ void __launch_bounds__(256)
lra_degrid_po_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                     const float* __restrict__ slabs, const float2* __restrict__ grid, const float* __restrict__ tau,
                     const float2* vis_in, float2* vis_out, int nchan, int nterms, int nx, int ny, int tile_x, lra_po_args po) {
  __shared__ float2 phs[8][2 * 129];
  const long long n = (long long)counters[0];
  const size_t plane = (size_t)nx * ny;
  const int lane = threadIdx.x & 31;
  float2* ph = phs[threadIdx.x >> 5];
  const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long i = warp0; i < n; i += nwarps) {
    const lra_rec r = rec[i];
    const int ix = r.x & 0xffff, iy = r.x >> 16, S = r.w & 0xff, h = (S - 1) >> 1;
    const float2* slab = reinterpret_cast<const float2*>(slabs + ((size_t)r.y << 2));
    const unsigned k = r.z;
    const int c = (int)(k % (unsigned)nchan);
    __syncwarp();
    const bool ok = lra_po_phasors(po, (long long)(k / (unsigned)nchan), ix, iy, S, nx, ny, ph, lane, 32);
    __syncwarp();
    if (!ok) continue;   // the init kernel left vis_in (or 0) there
    float tw[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) tw[t] = (t < nterms) ? (tau ? tau[c * nterms + t] : 1.0f) : 0.f;
    float2 acc[NC];
#pragma unroll
    for (int p = 0; p < NC; ++p) acc[p] = make_float2(0.f, 0.f);
    const float2* g0 = grid + (size_t)(iy - h) * nx + (ix - h);
    for (int j = 0; j < S; ++j) {
      const float2 b = ph[S + j];
      for (int ii = lane; ii < S; ii += 32) {
        const float2 c0 = slab[lra_tap_index(S, tile_x, j, ii)];
        const float2 a = ph[ii];
        const float2 f = make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
        const float2 cf = make_float2(c0.x * f.x - c0.y * f.y, c0.x * f.y + c0.y * f.x);
        const float2* gp = g0 + (size_t)j * nx + ii;
#pragma unroll
        for (int p = 0; p < NC; ++p) {
          float2 gs = make_float2(0.f, 0.f);
          for (int t = 0; t < nterms; ++t) {
            const float2 g = gp[(size_t)(t * NC + p) * plane];
            gs.x = fmaf(tw[t], g.x, gs.x);
            gs.y = fmaf(tw[t], g.y, gs.y);
          }
          // conj(cf) * gs
          acc[p].x = fmaf(cf.x, gs.x, acc[p].x);
          acc[p].x = fmaf(cf.y, gs.y, acc[p].x);
          acc[p].y = fmaf(cf.x, gs.y, acc[p].y);
          acc[p].y = fmaf(-cf.y, gs.x, acc[p].y);
        }
      }
    }
#pragma unroll
    for (int p = 0; p < NC; ++p)
      for (int o = 16; o > 0; o >>= 1) {
        acc[p].x += __shfl_xor_sync(0xffffffffu, acc[p].x, o);
        acc[p].y += __shfl_xor_sync(0xffffffffu, acc[p].y, o);
      }
    if (lane == 0) {
#pragma unroll
      for (int p = 0; p < NC; ++p) {
        float2 o = acc[p];
        if (vis_in) {
          const float2 vi = vis_in[(size_t)k * NC + p];
          o = make_float2(vi.x - acc[p].x, vi.y - acc[p].y);
        }
        vis_out[(size_t)k * NC + p] = o;
      }
    }
  }
}

__global__ void __launch_bounds__(256)
lra_copy_or_zero_kernel(const float2* __restrict__ src, float2* __restrict__ dst, long long n) {
  for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n; i += gridDim.x * 256ll)
    dst[i] = src ? src[i] : make_float2(0.f, 0.f);
}

// column q of [n][ncorr] arrays -> dense [n]
__global__ void __launch_bounds__(256)
lra_corr_gather_kernel(const float2* __restrict__ vis, const float* __restrict__ wt, int ncorr, int q, long long n,
                       float2* __restrict__ vis1, float* __restrict__ wt1) {
  for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n; i += gridDim.x * 256ll) {
    vis1[i] = vis[i * ncorr + q];
    if (wt) wt1[i] = wt[i * ncorr + q];
  }
}

// out[i][q] += sign * v1[i]
__global__ void __launch_bounds__(256)
lra_corr_add_kernel(const float2* __restrict__ v1, int ncorr, int q, long long n, float sign, float2* __restrict__ out) {
  for (long long i = blockIdx.x * 256ll + threadIdx.x; i < n; i += gridDim.x * 256ll) {
    const float2 v = v1[i];
    float2 o = out[i * ncorr + q];
    o.x += sign * v.x;
    o.y += sign * v.y;
    out[i * ncorr + q] = o;
  }
}

int lra_awp_reserve(lra_plan* p, size_t bytes) {
  if (p->awp_bytes >= bytes) return LRA_OK;
  if (p->awp_buf) { LRA_CUDA(p, cudaStreamSynchronize(p->stream)); cudaFree(p->awp_buf); p->awp_buf = nullptr; p->awp_bytes = 0; }
  LRA_CUDA(p, cudaMalloc(&p->awp_buf, bytes));
  p->awp_bytes = bytes;
  return LRA_OK;
}

int lra_po_scratch(lra_plan* p) {
  if (p->po_scratch) return LRA_OK;
  LRA_CUDA(p, cudaMalloc(&p->po_scratch, (size_t)p->ncorr * p->nterms * p->nx * p->ny * sizeof(float2)));
  return LRA_OK;
}

bool lra_po_valid(int n_po, const double* t) {
  if (n_po < 1 || n_po > (1 << 20) || !t) return false;
  for (int e = 0; e < 3 * n_po; ++e)
    if (!(t[e] == t[e]) || t[e] > 1e300 || t[e] < -1e300) return false;
  return true;
}

int lra_gradient(lra_plan* p, const float2* src, double f, double dl, double dm, bool conjugate, bool accumulate, float2* dst) {
  int rc = lra_awp_reserve(p, (size_t)(p->nx + p->ny) * sizeof(float2) + 4096);
  if (rc != LRA_OK) return rc;
  float2* tab = (float2*)p->awp_buf;
  const double sgn = conjugate ? -1.0 : 1.0;
  lra_gradient_table_kernel<<<(p->nx + p->ny + 255) / 256, 256, 0, p->stream>>>(tab, p->nx, p->ny, sgn * dl / p->scale_u,
                                                                                 sgn * dm / p->scale_v, f);
  LRA_LAUNCH_CHECK(p);
  const long long n = (long long)p->ncorr * p->nterms * p->nx * p->ny;
  const int blocks = (int)std::min<long long>((n + 255) / 256, (long long)p->sm_count * 16);
  if (accumulate) lra_phase_gradient_kernel<true><<<blocks, 256, 0, p->stream>>>(src, tab, dst, p->nx, p->ny, n);
  else lra_phase_gradient_kernel<false><<<blocks, 256, 0, p->stream>>>(src, tab, dst, p->nx, p->ny, n);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

// uploads the table behind the gradient phasors in awp_buf; -> device pointer
int lra_po_upload(lra_plan* p, int n_po, const double* table, const double** d_table) {
  const size_t off = ((size_t)(p->nx + p->ny) * sizeof(float2) + 4095) & ~(size_t)4095;
  int rc = lra_awp_reserve(p, off + (size_t)3 * n_po * sizeof(double));
  if (rc != LRA_OK) return rc;
  double* d = (double*)((char*)p->awp_buf + off);
  LRA_CUDA(p, cudaMemcpyAsync(d, table, (size_t)3 * n_po * sizeof(double), cudaMemcpyHostToDevice, p->stream));
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));   // the caller's table may be a temporary
  *d_table = d;
  return LRA_OK;
}

int lra_grid_po_impl(lra_plan* p, const float2* vis, const float* wt, const float* tau, int n_po, const double* table,
                     const int32_t* po_index, float2* grid, double* sumwt) {
  if (p->npoints == 0) return LRA_OK;
  if (!po_index) {   // one entry for every row: the tiled kernels, then the gradient on the whole grid
    int rc = lra_po_scratch(p);
    if (rc != LRA_OK) return rc;
    LRA_CUDA(p, cudaMemsetAsync(p->po_scratch, 0, (size_t)p->ncorr * p->nterms * p->nx * p->ny * sizeof(float2), p->stream));
    rc = lra_grid_impl(p, vis, wt, tau, p->po_scratch, sumwt);
    if (rc != LRA_OK) return rc;
    return lra_gradient(p, p->po_scratch, table[0], table[1], table[2], false, true, grid);
  }
  const double* d_table;
  int rc = lra_po_upload(p, n_po, table, &d_table);
  if (rc != LRA_OK) return rc;
  if (sumwt) { rc = lra_sumwt_launch(p, wt, tau, sumwt); if (rc != LRA_OK) return rc; }
  const lra_po_args po = {d_table, po_index, n_po, 1.0 / p->scale_u, 1.0 / p->scale_v};
  lra_grid_po_kernel<<<p->sm_count * 16, 256, 0, p->stream>>>(p->rec, p->counters, p->slabs, vis, wt, tau, p->nchan, p->ncorr,
                                                              p->nterms, p->nx, p->ny, p->tile_x, po, grid);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

int lra_degrid_po_impl(lra_plan* p, const float2* grid, const float* tau, int n_po, const double* table,
                       const int32_t* po_index, const float2* vis_in, float2* vis_out) {
  if (p->npoints == 0) return LRA_OK;
  if (!po_index) {   // conj(c f e^{i ph}) G = conj(c) (f e^{-i ph} G)
    int rc = lra_po_scratch(p);
    if (rc != LRA_OK) return rc;
    rc = lra_gradient(p, grid, table[0], table[1], table[2], true, false, p->po_scratch);
    if (rc != LRA_OK) return rc;
    return lra_degrid_impl(p, p->po_scratch, tau, vis_in, vis_out);
  }
  const double* d_table;
  int rc = lra_po_upload(p, n_po, table, &d_table);
  if (rc != LRA_OK) return rc;
  const long long nsamples = p->npoints * (long long)p->ncorr;
  if (vis_in != vis_out) {
    lra_copy_or_zero_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(vis_in, vis_out, nsamples);
    LRA_LAUNCH_CHECK(p);
  }
  const lra_po_args po = {d_table, po_index, n_po, 1.0 / p->scale_u, 1.0 / p->scale_v};
  const int blocks = p->sm_count * 8;
#define LRA_DG(NC) lra_degrid_po_kernel<NC><<<blocks, 256, 0, p->stream>>>(p->rec, p->counters, p->slabs, grid, tau, vis_in, \
                                                                           vis_out, p->nchan, p->nterms, p->nx, p->ny, p->tile_x, po)
  switch (p->ncorr) {
    case 1: LRA_DG(1); break;
    case 2: LRA_DG(2); break;
    case 3: LRA_DG(3); break;
    default: LRA_DG(4); break;
  }
#undef LRA_DG
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

}  // namespace

extern "C" int lra_phase_gradient(lra_plan* p, const void* src, double f, double dl, double dm, int32_t conjugate,
                                  int32_t accumulate, void* dst) {
  if (!p || !src || !dst || !(f == f) || !(dl == dl) || !(dm == dm)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_gradient(p, (const float2*)src, f, dl, dm, conjugate != 0, accumulate != 0, (float2*)dst);
}

extern "C" int lra_grid_po(lra_plan* p, const void* vis, const float* wt, const float* tau, int32_t n_po,
                           const double* po_table, const int32_t* po_index, void* grid, double* sumwt) {
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  if (!grid || (p->npoints > 0 && (!vis || !wt)) || !lra_po_valid(n_po, po_table)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_grid_po_impl(p, (const float2*)vis, wt, tau, n_po, po_table, po_index, (float2*)grid, sumwt);
}

extern "C" int lra_degrid_po(lra_plan* p, const void* grid, const float* tau, int32_t n_po, const double* po_table,
                             const int32_t* po_index, const void* vis_in, void* vis_out) {
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  if (!grid || (p->npoints > 0 && !vis_out) || !lra_po_valid(n_po, po_table)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_degrid_po_impl(p, (const float2*)grid, tau, n_po, po_table, po_index, (const float2*)vis_in, (float2*)vis_out);
}

// Mueller elements: plan with ncorr = nterms = 1; grid [ngrid][ny][nx], sumwt [ngrid]
static int lra_mueller_check(const lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                             int32_t n_elem, const int32_t* eg, const int32_t* ec, const int32_t* const* cfi, int32_t ncorr_vis,
                             int32_t ngrid, int32_t n_po, const double* po_table) {
  if (!p || p->ncorr != 1 || p->nterms != 1 || nrow < 0 || nchan < 1 || (nrow > 0 && !uvw) || !freq) return LRA_EINVAL;
  if (n_elem < 1 || n_elem > 16 || !eg || !ec || !cfi || ncorr_vis < 1 || ncorr_vis > 4 || ngrid < 1 || ngrid > 4) return LRA_EINVAL;
  for (int e = 0; e < n_elem; ++e)
    if (eg[e] < 0 || eg[e] >= ngrid || ec[e] < 0 || ec[e] >= ncorr_vis) return LRA_EINVAL;
  if (n_po != 0 && !lra_po_valid(n_po, po_table)) return LRA_EINVAL;
  if (nrow * (int64_t)nchan >= ((int64_t)1 << 31)) return LRA_EINVAL;
  return LRA_OK;
}

extern "C" int lra_grid_mueller(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq_hz,
                                int32_t n_elem, const int32_t* elem_grid, const int32_t* elem_corr,
                                const int32_t* const* cf_index, int32_t ncorr_vis, const void* vis, const float* wt,
                                const float* tau, int32_t n_po, const double* po_table, const int32_t* po_index,
                                int32_t ngrid, void* grid, double* sumwt) {
  int rc = lra_mueller_check(p, nrow, nchan, uvw, freq_hz, n_elem, elem_grid, elem_corr, cf_index, ncorr_vis, ngrid, n_po, po_table);
  if (rc != LRA_OK) return rc;
  if (!grid || (nrow > 0 && (!vis || !wt))) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  const long long n = nrow * (long long)nchan;
  float2* vis1 = nullptr;
  float* wt1 = nullptr;
  if (n > 0) {
    LRA_CUDA(p, cudaMalloc(&vis1, (size_t)n * (sizeof(float2) + sizeof(float))));
    wt1 = (float*)(vis1 + n);
  }
  const size_t plane = (size_t)p->nx * p->ny;
  for (int e = 0; e < n_elem && rc == LRA_OK; ++e) {
    rc = lra_bin_impl(p, nrow, nchan, uvw, freq_hz, cf_index[e]);
    if (rc != LRA_OK || n == 0) continue;
    lra_corr_gather_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>((const float2*)vis, wt, ncorr_vis, elem_corr[e], n, vis1, wt1);
    p->launches++;
    float2* g = (float2*)grid + (size_t)elem_grid[e] * plane;
    double* sw = (sumwt && elem_grid[e] == elem_corr[e]) ? sumwt + elem_grid[e] : nullptr;   // diagonal elements only [R29]
    rc = n_po ? lra_grid_po_impl(p, vis1, wt1, tau, n_po, po_table, po_index, g, sw) : lra_grid_impl(p, vis1, wt1, tau, g, sw);
  }
  if (vis1) { cudaStreamSynchronize(p->stream); cudaFree(vis1); }
  return rc;
}

extern "C" int lra_degrid_mueller(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq_hz,
                                  int32_t n_elem, const int32_t* elem_grid, const int32_t* elem_corr,
                                  const int32_t* const* cf_index, int32_t ncorr_vis, int32_t ngrid, const void* grid,
                                  const float* tau, int32_t n_po, const double* po_table, const int32_t* po_index,
                                  const void* vis_in, void* vis_out) {
  int rc = lra_mueller_check(p, nrow, nchan, uvw, freq_hz, n_elem, elem_grid, elem_corr, cf_index, ncorr_vis, ngrid, n_po, po_table);
  if (rc != LRA_OK) return rc;
  if (!grid || (nrow > 0 && !vis_out)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  const long long n = nrow * (long long)nchan;
  if (n == 0) return LRA_OK;
  float2* v1 = nullptr;
  LRA_CUDA(p, cudaMalloc(&v1, (size_t)n * sizeof(float2)));
  if (vis_in != vis_out) {
    lra_copy_or_zero_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>((const float2*)vis_in, (float2*)vis_out, n * ncorr_vis);
    p->launches++;
  }
  const size_t plane = (size_t)p->nx * p->ny;
  for (int e = 0; e < n_elem && rc == LRA_OK; ++e) {
    rc = lra_bin_impl(p, nrow, nchan, uvw, freq_hz, cf_index[e]);
    if (rc != LRA_OK) break;
    const float2* g = (const float2*)grid + (size_t)elem_grid[e] * plane;
    rc = n_po ? lra_degrid_po_impl(p, g, tau, n_po, po_table, po_index, nullptr, v1) : lra_degrid_impl(p, g, tau, nullptr, v1);
    if (rc != LRA_OK) break;
    lra_corr_add_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(v1, ncorr_vis, elem_corr[e], n, vis_in ? -1.f : 1.f, (float2*)vis_out);
    p->launches++;
  }
  cudaStreamSynchronize(p->stream);
  cudaFree(v1);
  return rc;
}

// ---- lra_phase_gradient_static: the phase gradient for callers that must not allocate -----------------------------------
// Same two kernels as lra_phase_gradient; the phasor table tab[nx + ny] lives in a file-scope device array instead of the
// plan's awp_buf, so the call needs no plan and issues no cudaMalloc / cudaFree (graph capture, serving loops).  Every
// GPU that loads liblra.so holds LRA_STATIC_MAX_AXES * 8 bytes = 512 KiB for it until the process exits.  The array is
// shared by all calls on a device: each call rewrites entries [0, nx + ny) before it reads them (nothing has to start at
// zero), and two calls whose kernels overlap on the GPU (different streams, no dependency) race on it.
static __device__ __align__(256) float2 lra_static_tab[LRA_STATIC_MAX_AXES];

namespace {

constexpr int LRA_STATIC_MAX_DEVICES = 64;
struct lra_static_device { float2* tab; int sm_count; };
lra_static_device lra_static_dev[LRA_STATIC_MAX_DEVICES];   // tab == nullptr: not resolved yet
std::mutex lra_static_mutex;
thread_local char lra_static_error[256] = "";

int lra_static_fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(lra_static_error, sizeof(lra_static_error), fmt, ap);
  va_end(ap);
  return code;
}

// In host code `lra_static_tab` is a host-side handle, not a device address: resolve it once per device, with that device
// current, and hand the resolved pointer to the kernels.
int lra_static_resolve(int device, lra_static_device* out) {
  std::lock_guard<std::mutex> lock(lra_static_mutex);
  lra_static_device& d = lra_static_dev[device];
  if (!d.tab) {
    float2* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&ptr, lra_static_tab);
    if (e != cudaSuccess || !ptr)
      return lra_static_fail(LRA_ECUDA, "cudaGetSymbolAddress(lra_static_tab) on device %d: %s", device, cudaGetErrorString(e));
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess || sms < 1)
      return lra_static_fail(LRA_ECUDA, "cudaDeviceGetAttribute(sm count) on device %d: %s", device, cudaGetErrorString(e));
    d.sm_count = sms;
    d.tab = ptr;
  }
  *out = d;
  return LRA_OK;
}

}  // namespace

extern "C" int lra_phase_gradient_static(int32_t nx, int32_t ny, int32_t nplanes, double scale_u, double scale_v,
                                         const void* src, double f, double dl, double dm, int32_t conjugate,
                                         int32_t accumulate, void* dst, void* stream) {
  lra_static_error[0] = 0;
  if (!src || !dst) return lra_static_fail(LRA_EINVAL, "lra_phase_gradient_static: src and dst must not be NULL");
  if (nx < 1 || ny < 1 || nplanes < 1)
    return lra_static_fail(LRA_EINVAL, "lra_phase_gradient_static: nx = %d, ny = %d, nplanes = %d must be >= 1", nx, ny, nplanes);
  if ((long long)nx + ny > LRA_STATIC_MAX_AXES)
    return lra_static_fail(LRA_EINVAL, "lra_phase_gradient_static: nx + ny = %lld exceeds the static table of LRA_STATIC_MAX_AXES = %d "
                           "entries; use lra_phase_gradient (plan-owned scratch) for larger grids", (long long)nx + ny, LRA_STATIC_MAX_AXES);
  if (!(f == f) || !(dl == dl) || !(dm == dm) || !(scale_u == scale_u) || !(scale_v == scale_v) || scale_u == 0.0 || scale_v == 0.0)
    return lra_static_fail(LRA_EINVAL, "lra_phase_gradient_static: f, dl, dm must be numbers and scale_u, scale_v non-zero");
  int device = -1;
  cudaError_t e = cudaGetDevice(&device);
  if (e != cudaSuccess) return lra_static_fail(LRA_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (device < 0 || device >= LRA_STATIC_MAX_DEVICES)
    return lra_static_fail(LRA_EINVAL, "lra_phase_gradient_static: device ordinal %d not below %d", device, LRA_STATIC_MAX_DEVICES);
  lra_static_device d;
  int rc = lra_static_resolve(device, &d);
  if (rc != LRA_OK) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  const double sgn = conjugate ? -1.0 : 1.0;
  lra_gradient_table_kernel<<<(nx + ny + 255) / 256, 256, 0, s>>>(d.tab, nx, ny, sgn * dl / scale_u, sgn * dm / scale_v, f);
  e = cudaGetLastError();
  if (e != cudaSuccess) return lra_static_fail(LRA_ECUDA, "lra_gradient_table_kernel launch: %s", cudaGetErrorString(e));
  const long long n = (long long)nplanes * nx * ny;
  const int blocks = (int)std::min<long long>((n + 255) / 256, (long long)d.sm_count * 16);
  if (accumulate) lra_phase_gradient_kernel<true><<<blocks, 256, 0, s>>>((const float2*)src, d.tab, (float2*)dst, nx, ny, n);
  else lra_phase_gradient_kernel<false><<<blocks, 256, 0, s>>>((const float2*)src, d.tab, (float2*)dst, nx, ny, n);
  e = cudaGetLastError();
  if (e != cudaSuccess) return lra_static_fail(LRA_ECUDA, "lra_phase_gradient_kernel launch: %s", cudaGetErrorString(e));
  return LRA_OK;
}

extern "C" const char* lra_static_last_error(void) { return lra_static_error; }
