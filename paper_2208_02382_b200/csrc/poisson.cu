// Free-space Poisson solve in the bunch rest frame ("the Poisson equation is solved in
// the bunch rest frame"), reading R19:
//   phi_a = (1/(4 pi eps0)) sum_b q_b G(r_a - r_b),  G(r) = 1/|r| (a != b),  G(0) = cell average of 1/r,
//   third-axis spacing dz' = gz * dz;  E = -grad phi by centred (faces: one-sided) differences.
// The open-boundary sum is a linear convolution, evaluated exactly (up to rounding) by Hockney's zero-padding: rho is
// embedded in a (2nx, 2ny, 2nz) box, transformed (cuFFT D2Z -- a library FFT is a step of the method, like the oracle's
// direct sum is a loop), multiplied by the transform of the Green table, transformed back, and the physical octant is kept.
// Everything around the two FFTs is this file's kernels: octant copy into a box zeroed once, Green table, spectral multiply (the table is even in every
// index, so its transform is real and only the real part is stored), and one pass that extracts phi and writes -grad phi into the
// 32-byte node records bt_gather_kick reads.  The transformed Green table is cached per (grid, gz).
#include "bt_internal.h"

#include <cufft.h>
#include <math.h>

namespace bt {

static const double kEps0 = 8.8541878128e-12;
static const double kPiP = 3.14159265358979323846264338327950288;

#define BT_CUFFT_TRY(expr)                                                                              \
    do {                                                                                                \
        cufftResult _r = (expr);                                                                        \
        if (_r != CUFFT_SUCCESS) return ::bt::fail(BT_ERR_CUDA, std::string(#expr) + ": cuFFT error " + std::to_string((int)_r)); \
    } while (0)

// ---- host: the self term, (1/V) int_cell 1/r dV, from the primitive F of 1/r (d^3F/dxdydz = 1/r) ---------------------
static long double box_primitive(long double x, long double y, long double z) {
    const long double r = sqrtl(x * x + y * y + z * z);
    long double f = 0.0L;
    if (x > 0 && y > 0 && z > 0)
        f -= 0.5L * (x * x * atanl(y * z / (x * r)) + y * y * atanl(x * z / (y * r)) + z * z * atanl(x * y / (z * r)));
    if (x > 0 && y > 0) f += x * y * logl(z + r);
    if (y > 0 && z > 0) f += y * z * logl(x + r);
    if (x > 0 && z > 0) f += x * z * logl(y + r);
    return f;
}
static double green_self_term(double dx, double dy, double dz) {
    const long double a = 0.5L * dx, b = 0.5L * dy, c = 0.5L * dz;
    // one octant: F(a,b,c) - F(0,b,c) - F(a,0,c) - F(a,b,0) (the terms with two or three zeros vanish); 8 octants / volume
    const long double oct = box_primitive(a, b, c) - box_primitive(0, b, c) - box_primitive(a, 0, c) - box_primitive(a, b, 0);
    return (double)(oct / (a * b * c));
}

// ---- kernels ---------------------------------------------------------------------------------------------------------
struct PadDims {
    int nx, ny, nz, mx, my, mz;  // physical and padded (m = 2n) node counts
};

// Green table on the padded box: index i stands for the offset i (i < n) or i - m (i > n); i == n is never used.
__global__ void __launch_bounds__(256) green_table_kernel(double *__restrict__ g, PadDims p, double dx, double dy, double dz, double g0) {
    const long long total = (long long)p.mx * p.my * p.mz;
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < total; a += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(a % p.mx), j = (int)((a / p.mx) % p.my), k = (int)(a / ((long long)p.mx * p.my));
        const int oi = i <= p.nx ? i : i - p.mx, oj = j <= p.ny ? j : j - p.my, ok = k <= p.nz ? k : k - p.mz;
        double v;
        if (i == p.nx || j == p.ny || k == p.nz) v = 0.0;
        else if (oi == 0 && oj == 0 && ok == 0) v = g0;
        else {
            const double rx = oi * dx, ry = oj * dy, rz = ok * dz;
            v = 1.0 / sqrt(rx * rx + ry * ry + rz * rz);
        }
        g[a] = v;
    }
}

__global__ void __launch_bounds__(256) real_part_kernel(const cufftDoubleComplex *__restrict__ spec, double *__restrict__ re, long long n) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) re[a] = spec[a].x;
}

// rho -> the physical octant of the padded input box (the other 7/8 of the box were zeroed once and are never written)
__global__ void __launch_bounds__(256) copy_octant_kernel(const double *__restrict__ rho, double *__restrict__ pad, PadDims p) {
    const long long total = (long long)p.nx * p.ny * p.nz;
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < total; a += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(a % p.nx), j = (int)((a / p.nx) % p.ny), k = (int)(a / ((long long)p.nx * p.ny));
        pad[((long long)k * p.my + j) * p.mx + i] = rho[a];
    }
}

__global__ void __launch_bounds__(256) spectral_multiply_kernel(cufftDoubleComplex *__restrict__ spec, const double *__restrict__ ghat,
                                                                long long n, double scale) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const double s = ghat[a] * scale;
        cufftDoubleComplex v = spec[a];
        v.x *= s;
        v.y *= s;
        spec[a] = v;
    }
}

// The physical octant of the padded potential -> phi, and E = -grad phi -> node records (Ex, Ey, Ez, 0): centred
// differences inside, one-sided first-order at the faces.  Reads the padded box directly (strides mx, mx*my).
__global__ void __launch_bounds__(256) gradient_kernel(const double *__restrict__ pad, double *__restrict__ phi, double4 *__restrict__ field,
                                                       PadDims p, double dx, double dy, double dz) {
    const long long total = (long long)p.nx * p.ny * p.nz;
    const long long sy = p.mx, sz = (long long)p.mx * p.my;
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < total; a += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(a % p.nx), j = (int)((a / p.nx) % p.ny), k = (int)(a / ((long long)p.nx * p.ny));
        const double *q = pad + ((long long)k * p.my + j) * p.mx + i;
        const double c = q[0];
        const double gx = i == 0 ? (q[1] - c) / dx : i == p.nx - 1 ? (c - q[-1]) / dx : (q[1] - q[-1]) / (2.0 * dx);
        const double gy = j == 0 ? (q[sy] - c) / dy : j == p.ny - 1 ? (c - q[-sy]) / dy : (q[sy] - q[-sy]) / (2.0 * dy);
        const double gzv = k == 0 ? (q[sz] - c) / dz : k == p.nz - 1 ? (c - q[-sz]) / dz : (q[sz] - q[-sz]) / (2.0 * dz);
        phi[a] = c;
        field[a] = make_double4(-gx, -gy, -gzv, 0.0);
    }
}

__global__ void __launch_bounds__(256) field_unpack_kernel(const double4 *__restrict__ field, long long nn, double *__restrict__ ex,
                                                           double *__restrict__ ey, double *__restrict__ ez) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a < nn) {
        const double4 v = field[a];
        ex[a] = v.x, ey[a] = v.y, ez[a] = v.z;
    }
}

// ---- host side -------------------------------------------------------------------------------------------------------
// The 3-D transforms are done as a batch of 2-D transforms over (y, x) for the planes that matter plus one strided 1-D pass
// over z: rho is zero on the planes z >= nz of the padded box and only the planes z < nz of the result are used, so both the
// forward and the inverse (y, x) passes run on nz instead of 2 nz planes -- a pruned FFT, a third of the work saved.
struct PoissonState {
    cufftHandle fwd2d = 0, zpass = 0, inv2d = 0;
    bool plans = false;
    double *in2d = nullptr;                // (nz, 2ny, 2nx) reals: rho in x < nx, y < ny; zeros elsewhere (zeroed once)
    cufftDoubleComplex *half = nullptr;    // (2nz, 2ny, nx + 1): the (y, x) transforms of the planes z < nz; planes z >= nz stay zero
    cufftDoubleComplex *spec = nullptr;    // (2nz, 2ny, nx + 1): full spectrum (z pass out of place, so `half` keeps its zeros)
    double *out2d = nullptr;               // (nz, 2ny, 2nx) reals: the potential on the planes z < nz of the padded box
    double *ghat = nullptr;                // real part of the Green table's transform, same shape as spec
    double ghat_gz = 0.0;                  // gz the cached table was built for (0 = none)
};

static int grid_1d(long long n) {
    long long b = (n + 255) / 256;
    return (int)(b > 148 * 32 ? 148 * 32 : b);
}

void poisson_free(Grid *g) {
    PoissonState *st = static_cast<PoissonState *>(g->poisson);
    if (!st) return;
    if (st->plans) {
        cufftDestroy(st->fwd2d);
        cufftDestroy(st->zpass);
        cufftDestroy(st->inv2d);
    }
    if (st->in2d) cudaFree(st->in2d);
    if (st->half) cudaFree(st->half);
    if (st->spec) cudaFree(st->spec);
    if (st->out2d) cudaFree(st->out2d);
    if (st->ghat) cudaFree(st->ghat);
    delete st;
    g->poisson = nullptr;
}

// Transform of the (dense) Green table: a plain 3-D D2Z with a temporary plan and buffer, once per gz.
static int build_green_transform(PoissonState *st, const PadDims &p, double dx, double dy, double dz, cudaStream_t stream) {
    const long long nreal = (long long)p.mx * p.my * p.mz;
    const long long nspec = (long long)p.mz * p.my * (p.mx / 2 + 1);
    double *table = nullptr;
    BT_CUDA_TRY(cudaMalloc(&table, (size_t)nreal * sizeof(double)));
    cufftHandle plan3d = 0;
    cufftResult r = cufftPlan3d(&plan3d, p.mz, p.my, p.mx, CUFFT_D2Z);
    if (r == CUFFT_SUCCESS) r = cufftSetStream(plan3d, stream);
    if (r == CUFFT_SUCCESS) {
        green_table_kernel<<<grid_1d(nreal), 256, 0, stream>>>(table, p, dx, dy, dz, green_self_term(dx, dy, dz));
        r = cufftExecD2Z(plan3d, table, st->spec);
    }
    if (r == CUFFT_SUCCESS) real_part_kernel<<<grid_1d(nspec), 256, 0, stream>>>(st->spec, st->ghat, nspec);
    cudaStreamSynchronize(stream);  // the temporaries go away
    if (plan3d) cufftDestroy(plan3d);
    cudaFree(table);
    if (r != CUFFT_SUCCESS) return fail(BT_ERR_CUDA, "bt_grid_solve_poisson: cuFFT error " + std::to_string((int)r) + " while transforming the Green table");
    g_launch_count.fetch_add(2);
    return BT_OK;
}

int poisson_solve(Grid *g, double gz, cudaStream_t stream) {
    PadDims p;
    p.nx = g->nx, p.ny = g->ny, p.nz = g->nz;
    p.mx = 2 * g->nx, p.my = 2 * g->ny, p.mz = 2 * g->nz;
    const int hx = p.mx / 2 + 1;
    const long long nreal = (long long)p.mx * p.my * p.mz;
    const long long nplane_r = (long long)p.my * p.mx, nplane_c = (long long)p.my * hx;
    const long long nspec = (long long)p.mz * nplane_c;
    PoissonState *st = static_cast<PoissonState *>(g->poisson);
    if (!st) {
        st = new (std::nothrow) PoissonState();
        if (!st) return fail(BT_ERR_OOM, "bt_grid_solve_poisson: host allocation failed");
        g->poisson = st;
    }
    if (!st->in2d) {
        BT_CUDA_TRY(cudaMalloc(&st->in2d, (size_t)(p.nz * nplane_r) * sizeof(double)));
        BT_CUDA_TRY(cudaMemsetAsync(st->in2d, 0, (size_t)(p.nz * nplane_r) * sizeof(double), stream));  // transforms are out of place: zeros persist
    }
    if (!st->half) {
        BT_CUDA_TRY(cudaMalloc(&st->half, (size_t)nspec * sizeof(cufftDoubleComplex)));
        BT_CUDA_TRY(cudaMemsetAsync(st->half, 0, (size_t)nspec * sizeof(cufftDoubleComplex), stream));
    }
    if (!st->out2d) BT_CUDA_TRY(cudaMalloc(&st->out2d, (size_t)(p.nz * nplane_r) * sizeof(double)));
    if (!st->spec) BT_CUDA_TRY(cudaMalloc(&st->spec, (size_t)nspec * sizeof(cufftDoubleComplex)));
    if (!st->ghat) BT_CUDA_TRY(cudaMalloc(&st->ghat, (size_t)nspec * sizeof(double)));
    if (!g->phi) BT_CUDA_TRY(cudaMalloc(&g->phi, (size_t)g->nn * sizeof(double)));
    if (!g->field) BT_CUDA_TRY(cudaMalloc(&g->field, (size_t)g->nn * 4 * sizeof(double)));
    if (!st->plans) {
        int n2[2] = {p.my, p.mx}, emb_r[2] = {p.my, p.mx}, emb_c[2] = {p.my, hx}, n1[1] = {p.mz}, emb_z[1] = {p.mz};
        BT_CUFFT_TRY(cufftPlanMany(&st->fwd2d, 2, n2, emb_r, 1, (int)nplane_r, emb_c, 1, (int)nplane_c, CUFFT_D2Z, p.nz));
        BT_CUFFT_TRY(cufftPlanMany(&st->zpass, 1, n1, emb_z, (int)nplane_c, 1, emb_z, (int)nplane_c, 1, CUFFT_Z2Z, (int)nplane_c));
        BT_CUFFT_TRY(cufftPlanMany(&st->inv2d, 2, n2, emb_c, 1, (int)nplane_c, emb_r, 1, (int)nplane_r, CUFFT_Z2D, p.nz));
        st->plans = true;
    }
    BT_CUFFT_TRY(cufftSetStream(st->fwd2d, stream));
    BT_CUFFT_TRY(cufftSetStream(st->zpass, stream));
    BT_CUFFT_TRY(cufftSetStream(st->inv2d, stream));
    const double dx = g->d[0], dy = g->d[1], dz = gz * g->d[2];
    if (st->ghat_gz != gz) {  // Green table for this grid and this gz: built and transformed once
        const int rc = build_green_transform(st, p, dx, dy, dz, stream);
        if (rc != BT_OK) return rc;
        st->ghat_gz = gz;
    }
    copy_octant_kernel<<<grid_1d(g->nn), 256, 0, stream>>>(g->rho, st->in2d, p);
    BT_CUFFT_TRY(cufftExecD2Z(st->fwd2d, st->in2d, st->half));                    // (y, x) on the planes z < nz
    BT_CUFFT_TRY(cufftExecZ2Z(st->zpass, st->half, st->spec, CUFFT_FORWARD));     // z
    const double scale = 1.0 / (4.0 * kPiP * kEps0) / (double)nreal;  // Coulomb constant and the unnormalised inverse FFT
    spectral_multiply_kernel<<<grid_1d(nspec), 256, 0, stream>>>(st->spec, st->ghat, nspec, scale);
    BT_CUFFT_TRY(cufftExecZ2Z(st->zpass, st->spec, st->spec, CUFFT_INVERSE));     // z, in place
    BT_CUFFT_TRY(cufftExecZ2D(st->inv2d, st->spec, st->out2d));                   // (y, x) on the planes z < nz
    gradient_kernel<<<grid_1d(g->nn), 256, 0, stream>>>(st->out2d, g->phi, reinterpret_cast<double4 *>(g->field), p, dx, dy, dz);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_grid_solve_poisson launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(3);
    return BT_OK;
}

int field_unpack(Grid *g, double *ex, double *ey, double *ez, cudaStream_t stream) {
    field_unpack_kernel<<<(int)((g->nn + 255) / 256), 256, 0, stream>>>(reinterpret_cast<const double4 *>(g->field), g->nn, ex, ey, ez);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_grid_download_field launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

}  // namespace bt
