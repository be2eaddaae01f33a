// pm.cu -- libhaccpm.so: HACC's long-range particle-mesh force, see
// include/haccpm.h.  Kernels: CIC deposit (float atomics), the spectral multiply that composes
// influence function, filter and Lanczos derivative ("one single Fourier transform",
// PAPER.md:157), CIC interpolation with the optional long-range kick.  FFTs: cuFFT (a plain
// library FFT).  Nothing here is shared with oracle/.
#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/haccpm.h"

struct haccpm_ctx {
    int ng = 0;
    float box_l = 0.f;
    int device = 0;
    int n_sms = 0;
    cudaStream_t stream = nullptr;
    cufftHandle r2c = 0, c2r = 0;
    bool plans = false;
    float *rho = nullptr;          // [ng^3] density (kept for haccpm_get_density)
    float *field[3] = {nullptr, nullptr, nullptr};  // [ng^3] each: a_x, a_y, a_z on the grid
    float4 *field4 = nullptr;      // [ng^3] {a_x, a_y, a_z, 0} per node: what k_pm_interp gathers
    cufftComplex *rho_k = nullptr; // [ng^2 (ng/2+1)]
    cufftComplex *work_k = nullptr;
    double *tab_e = nullptr;       // [ng] cos(t) - 5/64 cos(2t) + 1/1024 cos(4t)      (Eq. 5)
    double *tab_s = nullptr;       // [ng] exp(-t^2 sigma^2/4) [(2/t) sin(t/2)]^ns     (Eq. 6)
    double *tab_d = nullptr;       // [ng] (4/3) sin(t) - (1/6) sin(2t)                (Eq. 7)
    int *error_flag = nullptr;
};

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) & ~(kAlign - 1); }

struct Layout {
    size_t rho, field[3], field4, rho_k, work_k, tab_e, tab_s, tab_d, flag, total;
};

bool layout_for(int ng, Layout &l)
{
    if (ng < 4 || ng > 2048 || (ng & 1)) return false;
    const size_t n3 = (size_t)ng * ng * ng, nk = (size_t)ng * ng * (ng / 2 + 1);
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t at = o;
        o = align_up(o + bytes);
        return at;
    };
    l.rho = take(sizeof(float) * n3);
    for (int k = 0; k < 3; ++k) l.field[k] = take(sizeof(float) * n3);
    l.field4 = take(sizeof(float4) * n3);
    l.rho_k = take(sizeof(cufftComplex) * nk);
    l.work_k = take(sizeof(cufftComplex) * nk);
    l.tab_e = take(sizeof(double) * ng);
    l.tab_s = take(sizeof(double) * ng);
    l.tab_d = take(sizeof(double) * ng);
    l.flag = take(sizeof(int));
    l.total = o;
    return true;
}

class DeviceGuard {
public:
    explicit DeviceGuard(int want) : want_(want)
    {
        ok_ = cudaGetDevice(&prev_) == cudaSuccess;
        if (ok_ && prev_ != want_) ok_ = cudaSetDevice(want_) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (ok_ && prev_ != want_) cudaSetDevice(prev_);
    }
    bool ok() const { return ok_; }

private:
    int prev_ = 0, want_ = 0;
    bool ok_ = false;
};

// position -> (lower grid index, fraction) per dimension; wraps into [0, L); NaN/Inf -> bad
__device__ __forceinline__ void cic_coord(float p, float box_l, float inv_delta, int ng, int &i0,
                                          float &d, bool &bad)
{
    if (!(p >= 0.f && p < box_l)) {
        if (!isfinite(p)) {
            bad = true;
            p = 0.f;
        } else {
            p = p - box_l * floorf(p / box_l);
            if (!(p >= 0.f && p < box_l)) p = 0.f;
        }
    }
    const float u = p * inv_delta;
    const float f = floorf(u);
    i0 = min(max((int)f, 0), ng - 1);
    d = u - (float)i0;
}

__global__ void __launch_bounds__(256) k_pm_deposit(int64_t n, const float *__restrict__ x,
                                                    const float *__restrict__ y,
                                                    const float *__restrict__ z,
                                                    const float *__restrict__ mass, float box_l,
                                                    float inv_delta, float inv_vol, int ng,
                                                    float *__restrict__ rho, int *error_flag)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        int ix, iy, iz;
        float dx, dy, dz;
        cic_coord(__ldg(x + i), box_l, inv_delta, ng, ix, dx, bad);
        cic_coord(__ldg(y + i), box_l, inv_delta, ng, iy, dy, bad);
        cic_coord(__ldg(z + i), box_l, inv_delta, ng, iz, dz, bad);
        const float m = (mass ? __ldg(mass + i) : 1.f) * inv_vol;
        const int jx = (ix + 1 == ng) ? 0 : ix + 1, jy = (iy + 1 == ng) ? 0 : iy + 1,
                  jz = (iz + 1 == ng) ? 0 : iz + 1;
        const float wx[2] = {1.f - dx, dx}, wy[2] = {1.f - dy, dy}, wz[2] = {1.f - dz, dz};
        const int cx[2] = {ix, jx}, cy[2] = {iy, jy}, cz[2] = {iz, jz};
        // nodes iz and iz+1 are neighbours in memory: one 8-byte atomic for the pair when it
        // is 8-byte aligned (iz even; ng is even, so an even iz never wraps)
        const bool pair = (iz & 1) == 0;
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                float *row = rho + ((size_t)cx[a] * ng + cy[b]) * ng;
                const float w0 = m * wx[a] * wy[b] * wz[0], w1 = m * wx[a] * wy[b] * wz[1];
                if (pair) {
                    atomicAdd(reinterpret_cast<float2 *>(row + iz), make_float2(w0, w1));
                } else {
                    atomicAdd(row + iz, w0);
                    atomicAdd(row + jz, w1);
                }
            }
    }
    if (bad) *error_flag = HACCPM_EDATA;
}

// out(k) = -D_comp(k) * 4 pi G6(k) S(k) rho(k) / ng^3  (the 1/ng^3 of the inverse transform).
// The multiplier is real times -i: (re + i im) * (-i c) = c im - i c re.  Tables and the
// bracket of Eq. 5 (a difference of O(1) terms that is O(theta^2)) are in double.
__global__ void __launch_bounds__(256) k_pm_green(int ng, int comp, double scale,
                                                  const double *__restrict__ tab_e,
                                                  const double *__restrict__ tab_s,
                                                  const double *__restrict__ tab_d,
                                                  const cufftComplex *__restrict__ rho_k,
                                                  cufftComplex *__restrict__ out)
{
    const int nzh = ng / 2 + 1;
    const size_t total = (size_t)ng * ng * nzh;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int iz = (int)(e % nzh);
        const int iy = (int)((e / nzh) % ng);
        const int ix = (int)(e / ((size_t)nzh * ng));
        float c = 0.f;
        if (ix | iy | iz) {
            const double den = tab_e[ix] + tab_e[iy] + tab_e[iz] - 2835.0 / 1024.0;
            const double d = tab_d[comp == 0 ? ix : comp == 1 ? iy : iz];
            if (fabs(den) > 1e-14) c = (float)(scale * d * tab_s[ix] * tab_s[iy] * tab_s[iz] / den);
        }
        const cufftComplex r = rho_k[e];
        out[e] = make_float2(c * r.y, -c * r.x);
    }
}

// The three components side by side, 16 bytes per node: the 8 nodes of a particle's CIC cell
// are then 4 runs of 32 bytes (z and z+1 are neighbours in memory) holding all three
// components, instead of 3 x 4 runs in three grids.  Particles arrive in any order, so every
// run is a DRAM access of its own: 3.4x less traffic for the gather.
__global__ void __launch_bounds__(256) k_pm_pack(size_t n3, const float *__restrict__ fx,
                                                 const float *__restrict__ fy,
                                                 const float *__restrict__ fz,
                                                 float4 *__restrict__ out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n3; e += stride)
        out[e] = make_float4(fx[e], fy[e], fz[e], 0.f);
}

// CIC interpolation of the three components in one pass ("interpolated back to
// the particles"), with the optional long-range kick v += dt * a of Eq. 9.
__global__ void __launch_bounds__(256) k_pm_interp(int64_t n, const float *__restrict__ x,
                                                   const float *__restrict__ y,
                                                   const float *__restrict__ z, float box_l,
                                                   float inv_delta, int ng,
                                                   const float4 *__restrict__ field,
                                                   float *__restrict__ ax, float *__restrict__ ay,
                                                   float *__restrict__ az, float dt,
                                                   float *__restrict__ vx, float *__restrict__ vy,
                                                   float *__restrict__ vz)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        int ix, iy, iz;
        float dx, dy, dz;
        cic_coord(__ldg(x + i), box_l, inv_delta, ng, ix, dx, bad);
        cic_coord(__ldg(y + i), box_l, inv_delta, ng, iy, dy, bad);
        cic_coord(__ldg(z + i), box_l, inv_delta, ng, iz, dz, bad);
        const int jx = (ix + 1 == ng) ? 0 : ix + 1, jy = (iy + 1 == ng) ? 0 : iy + 1,
                  jz = (iz + 1 == ng) ? 0 : iz + 1;
        const float wx[2] = {1.f - dx, dx}, wy[2] = {1.f - dy, dy}, wz[2] = {1.f - dz, dz};
        const int cx[2] = {ix, jx}, cy[2] = {iy, jy}, cz[2] = {iz, jz};
        float4 f[8];   // all eight gathers in flight before the first use
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int q = 0; q < 2; ++q)
#pragma unroll
                for (int r = 0; r < 2; ++r)
                    f[4 * p + 2 * q + r] = __ldg(field + ((size_t)cx[p] * ng + cy[q]) * ng + cz[r]);
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int q = 0; q < 2; ++q)
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const float wgt = wx[p] * wy[q] * wz[r];
                    a0 = fmaf(wgt, f[4 * p + 2 * q + r].x, a0);
                    a1 = fmaf(wgt, f[4 * p + 2 * q + r].y, a1);
                    a2 = fmaf(wgt, f[4 * p + 2 * q + r].z, a2);
                }
        ax[i] = a0;
        ay[i] = a1;
        az[i] = a2;
        if (vx) {
            vx[i] = fmaf(dt, a0, vx[i]);
            vy[i] = fmaf(dt, a1, vy[i]);
            vz[i] = fmaf(dt, a2, vz[i]);
        }
    }
    (void)bad;   // a non-finite position was already flagged by the deposit
}

inline int grid_for(const haccpm_ctx *c, size_t n)
{
    const size_t want = (n + 255) / 256, cap = (size_t)c->n_sms * 16;
    return (int)(want < cap ? (want > 0 ? want : 1) : cap);
}

}  // namespace

extern "C" {

int haccpm_abi_version(void) { return 1; }

size_t haccpm_workspace_bytes(int ng)
{
    Layout l;
    return layout_for(ng, l) ? l.total : 0;
}

int haccpm_create(haccpm_ctx **out, int ng, float box_L, float sigma, int n_s, void *workspace,
                  size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return HACCPM_EINVAL;
    *out = nullptr;
    Layout l;
    if (!layout_for(ng, l)) return HACCPM_EINVAL;
    if (!(box_L > 0.f) || !std::isfinite(box_L) || !(sigma >= 0.f) || !std::isfinite(sigma) ||
        n_s < 0 || n_s > 16)
        return HACCPM_EINVAL;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1))) return HACCPM_EINVAL;
    if (workspace_bytes < l.total) return HACCPM_ENOMEM;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HACCPM_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCPM_ECUDA;
    haccpm_ctx *c = new (std::nothrow) haccpm_ctx();
    if (!c) return HACCPM_ENOMEM;
    c->ng = ng;
    c->box_l = box_L;
    c->device = dev;
    c->n_sms = sms;
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    char *w = static_cast<char *>(workspace);
    c->rho = reinterpret_cast<float *>(w + l.rho);
    for (int k = 0; k < 3; ++k) c->field[k] = reinterpret_cast<float *>(w + l.field[k]);
    c->field4 = reinterpret_cast<float4 *>(w + l.field4);
    c->rho_k = reinterpret_cast<cufftComplex *>(w + l.rho_k);
    c->work_k = reinterpret_cast<cufftComplex *>(w + l.work_k);
    c->tab_e = reinterpret_cast<double *>(w + l.tab_e);
    c->tab_s = reinterpret_cast<double *>(w + l.tab_s);
    c->tab_d = reinterpret_cast<double *>(w + l.tab_d);
    c->error_flag = reinterpret_cast<int *>(w + l.flag);
    // per-dimension tables in double: theta = 2 pi k / ng, k = index or index - ng
    std::vector<double> te(ng), ts(ng), td(ng);
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < ng; ++i) {
        const int k = (i <= ng / 2 - 1) ? i : i - ng;   // (index ng/2 is the Nyquist mode -ng/2)
        const double t = 2.0 * pi * (double)k / (double)ng;
        te[i] = std::cos(t) - (5.0 / 64.0) * std::cos(2.0 * t) + (1.0 / 1024.0) * std::cos(4.0 * t);
        const double sinc = (std::fabs(t) > 1e-12) ? (2.0 / t) * std::sin(t / 2.0) : 1.0;
        ts[i] = std::exp(-t * t * (double)sigma * (double)sigma / 4.0) * std::pow(sinc, n_s);
        td[i] = (4.0 / 3.0) * std::sin(t) - (1.0 / 6.0) * std::sin(2.0 * t);
    }
    bool ok = cudaMemcpy(c->tab_e, te.data(), sizeof(double) * ng, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(c->tab_s, ts.data(), sizeof(double) * ng, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(c->tab_d, td.data(), sizeof(double) * ng, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemset(c->error_flag, 0, sizeof(int)) == cudaSuccess;
    if (ok) {
        ok = cufftPlan3d(&c->r2c, ng, ng, ng, CUFFT_R2C) == CUFFT_SUCCESS;
        if (ok) {
            ok = cufftPlan3d(&c->c2r, ng, ng, ng, CUFFT_C2R) == CUFFT_SUCCESS;
            if (!ok) cufftDestroy(c->r2c);
        }
        if (ok) {
            c->plans = true;
            ok = cufftSetStream(c->r2c, c->stream) == CUFFT_SUCCESS &&
                 cufftSetStream(c->c2r, c->stream) == CUFFT_SUCCESS;
        }
    }
    if (!ok) {
        if (c->plans) {
            cufftDestroy(c->r2c);
            cufftDestroy(c->c2r);
        }
        delete c;
        return HACCPM_ECUDA;
    }
    *out = c;
    return HACCPM_OK;
}

int haccpm_destroy(haccpm_ctx *c)
{
    if (!c) return HACCPM_EINVAL;
    {
        DeviceGuard guard(c->device);
        if (guard.ok()) cudaStreamSynchronize(c->stream);
        if (c->plans) {
            cufftDestroy(c->r2c);
            cufftDestroy(c->c2r);
        }
    }
    delete c;
    return HACCPM_OK;
}

int hacc_lr_force(haccpm_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                  const float *mass, float *ax, float *ay, float *az, float dt, float *vx,
                  float *vy, float *vz)
{
    if (!c || n < 0 || !std::isfinite(dt)) return HACCPM_EINVAL;
    if (n > 0 && (!x || !y || !z || !ax || !ay || !az)) return HACCPM_EINVAL;
    const int nv = (vx != nullptr) + (vy != nullptr) + (vz != nullptr);
    if (nv != 0 && nv != 3) return HACCPM_EINVAL;
    DeviceGuard guard(c->device);
    if (!guard.ok()) return HACCPM_ECUDA;
    const int ng = c->ng;
    const size_t n3 = (size_t)ng * ng * ng, nk = (size_t)ng * ng * (ng / 2 + 1);
    const double delta = (double)c->box_l / ng;
    const float inv_delta = (float)(1.0 / delta), inv_vol = (float)(1.0 / (delta * delta * delta));
    cudaStream_t st = c->stream;
    if (cudaMemsetAsync(c->rho, 0, sizeof(float) * n3, st) != cudaSuccess) return HACCPM_ECUDA;
    if (n > 0)
        k_pm_deposit<<<grid_for(c, (size_t)n), 256, 0, st>>>(n, x, y, z, mass, c->box_l, inv_delta,
                                                             inv_vol, ng, c->rho, c->error_flag);
    if (cufftExecR2C(c->r2c, c->rho, c->rho_k) != CUFFT_SUCCESS) return HACCPM_ECUDA;
    // a(k) = -D 4 pi G6 S rho(k): -i * [dval/Delta] * 4 pi (45/128) Delta^2 / den * S, and the
    // 1/ng^3 of the unnormalised inverse transform
    const double scale = 4.0 * 3.14159265358979323846 * (45.0 / 128.0) * delta / (double)n3;
    for (int comp = 0; comp < 3; ++comp) {
        k_pm_green<<<grid_for(c, nk), 256, 0, st>>>(ng, comp, scale, c->tab_e, c->tab_s, c->tab_d,
                                                    c->rho_k, c->work_k);
        if (cufftExecC2R(c->c2r, c->work_k, c->field[comp]) != CUFFT_SUCCESS) return HACCPM_ECUDA;
    }
    if (n > 0) {
        k_pm_pack<<<grid_for(c, n3), 256, 0, st>>>(n3, c->field[0], c->field[1], c->field[2],
                                                   c->field4);
        k_pm_interp<<<grid_for(c, (size_t)n), 256, 0, st>>>(n, x, y, z, c->box_l, inv_delta, ng,
                                                            c->field4, ax, ay, az, dt, vx, vy, vz);
    }
    return cudaGetLastError() == cudaSuccess ? HACCPM_OK : HACCPM_ECUDA;
}

int haccpm_get_density(haccpm_ctx *c, const float **rho)
{
    if (!c || !rho) return HACCPM_EINVAL;
    *rho = c->rho;
    return HACCPM_OK;
}

int haccpm_sync(haccpm_ctx *c)
{
    if (!c) return HACCPM_EINVAL;
    DeviceGuard guard(c->device);
    if (!guard.ok()) return HACCPM_ECUDA;
    int flag = 0;
    if (cudaMemcpyAsync(&flag, c->error_flag, sizeof(flag), cudaMemcpyDeviceToHost, c->stream) !=
        cudaSuccess)
        return HACCPM_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HACCPM_ECUDA;
    if (flag != 0) {
        cudaMemsetAsync(c->error_flag, 0, sizeof(flag), c->stream);
        return flag;
    }
    return HACCPM_OK;
}

}  // extern "C"
