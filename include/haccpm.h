/*
 * haccpm.h -- C ABI of libhaccpm.so: HACC's long-range (particle-mesh) force on one B200.
 * Companion of haccsr.h (the short-range force); a separate library because it links cuFFT.
 *
 * What is computed (PAPER.md = arxiv 1410.2805, section 2.3):
 *   "The HACC long-range force solver uses only CIC mass deposition and force interpolation
 *    with a Gauss-sinc spectral filter ... a fourth-order Super-Lanczos spectral differentiator
 *    ... along with a sixth-order influence function"; "The 'Poisson-solve' in the
 *    HACC code is the composition of all the kernels above in one single Fourier transform ...
 *    each component of the field gradient requires an independent FFT":
 *
 *     rho(g)   = sum_p m_p W(x_p - g) / Delta^3                  CIC deposit, periodic
 *     a_i(k)   = -D_i(k) * 4 pi G6(k) * S(k) * rho(k)            Eqs. 7, 5, 6; G = 1; k = 0 dropped
 *     a_i(x_p) = sum_g W(x_p - g) a_i(g)                         CIC interpolation
 *
 *   theta_j = 2 pi k_j Delta / L;  G6 = (45/128) Delta^2 / [sum_j cos(theta_j) - (5/64) sum_j
 *   cos(2 theta_j) + (1/1024) sum_j cos(4 theta_j) - 2835/1024];  S = exp(-|theta|^2 sigma^2/4)
 *   prod_j [(2/theta_j) sin(theta_j/2)]^n_s;  D_i = i [(4/3) sin(theta_i) - (1/6) sin(2 theta_i)]
 *   / Delta.  Together with the short-range force of haccsr.h this closes the gravity loop:
 *   a_lr + a_sr is Newtonian (Fig. 3).
 *
 * Conventions as in haccsr.h: DEVICE pointers owned by the caller unless marked HOST; work is
 * enqueued on the stream given at creation; negative status on error; no CPU fallback.
 * Particle arrays are float32 SoA in the periodic box [0, L); positions outside are wrapped.
 * The arithmetic is float32 (cuFFT single precision); the three per-dimension kernel tables
 * are built in double on the host at creation.
 */
#ifndef HACCPM_H
#define HACCPM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct haccpm_ctx haccpm_ctx;

enum {
    HACCPM_OK = 0,
    HACCPM_EINVAL = -1, /* bad argument */
    HACCPM_ENOMEM = -3, /* workspace too small */
    HACCPM_ECUDA = -4,  /* CUDA / cuFFT error (including: no device) */
    HACCPM_EDATA = -5   /* NaN/Inf position seen on the device */
};

int haccpm_abi_version(void);

/* Bytes of device workspace for an ng^3 grid (0 for ng < 4, ng > 2048 or odd ng). */
size_t haccpm_workspace_bytes(int ng);

/*
 * Create a solver for an ng^3 grid over the periodic box of length box_L (Delta = box_L/ng;
 * HACC runs with Delta = 1 grid unit).  sigma (grid cells) and n_s are the filter parameters
 * of Eq. 6 (HACC: 0.8 and 3).  workspace: device, >= haccpm_workspace_bytes, 256-byte aligned.
 * The cuFFT plans (and their own work areas) are created here; nothing is allocated later.
 */
int haccpm_create(haccpm_ctx **out, int ng, float box_L, float sigma, int n_s, void *workspace,
                  size_t workspace_bytes, void *cuda_stream);
int haccpm_destroy(haccpm_ctx *ctx);

/*
 * hacc_lr_force -- long-range accelerations at the particle positions: deposit, one forward
 * FFT, and per component the spectral multiply, an inverse FFT and the interpolation.
 * x,y,z: length n; mass: length n or NULL (unit masses); ax,ay,az: length n, overwritten.
 * If vx,vy,vz are all non-NULL the long-range kick of Eq. 9 (M_lr) is fused into
 * the interpolation: v <- v + dt * a.
 */
int hacc_lr_force(haccpm_ctx *ctx, int64_t n, const float *x, const float *y, const float *z,
                  const float *mass, float *ax, float *ay, float *az, float dt, float *vx,
                  float *vy, float *vz);

/* Read-only view of the deposited density grid of the last call (ng^3 floats, z fastest). */
int haccpm_get_density(haccpm_ctx *ctx, const float **rho);

/* Stream synchronise + fetch (and clear) the device error flag. */
int haccpm_sync(haccpm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* HACCPM_H */
