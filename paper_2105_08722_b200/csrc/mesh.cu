// mesh.cu — the gridded estimator (eq. 36):
//
//   a^b_lm(s) = F^-1[ F[delta](k) F[Y_lm(r^) Theta^b(r)](k) ](s) / int dr Theta^b(r)                     eq. 36
//
// for a density field on a periodic G^3 mesh, then the same per-primary contraction (steps a5, a6) with one "primary"
// per mesh cell.  Discretised on the mesh (int dr -> h^3 sum over cells) this is eq. 34/35 for particles at the cell
// centres with weights delta h^3:  a(s) = (1/v_b) sum_{x != s} delta(x) h^3 Y_lm((x-s)^) Theta^b(|x-s|), a cyclic
// cross-correlation, evaluated here with cuFFT (a library FFT as a step of the path): per (bin, l, m >= 0) one kernel
// samples conj(Y_lm) Theta^b at the minimal-image lattice offsets, forward FFT, multiply with conj into F[delta h^3],
// inverse FFT, and the real / imaginary parts go straight into the a_lm tile layout of the contraction kernels
// ([group of 32 consecutive cells][component][bin][lane]).  The paper has no gridded code: the FFT route
// is its eq. 36, the tile layout and the contraction are this library's.
#include "device.cuh"

#include <cufft.h>

namespace {

constexpr int kT = 256;

__global__ void k_mesh_weights(const double *__restrict__ delta, size_t ncell, double h3, cufftDoubleComplex *__restrict__ fd,
                               double *__restrict__ gweights, size_t npad)
{
    const size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (c >= npad) return;
    const double w = c < ncell ? delta[c] * h3 : 0.0;
    gweights[c] = w;
    if (c < ncell) fd[c] = make_cuDoubleComplex(w, 0.0);
}

// kern[c] = conj(Y_lm(r^)) Theta^b(r) at the minimal-image offset of cell c from cell 0, r = h |offset|;
// Y_lm = sum_k ycoef[comp][k] z^k (x+iy)^m (tables.cpp), bins decided on r^2 against e_b^2 (R8, R9)
// blockIdx.y = field of the batch: (l, m >= 0) number j0 + blockIdx.y in the order l ascending, m ascending
__global__ void k_mesh_kernel(int G, double h, int j0, int nlm, int lmax, const double *__restrict__ ycoef, double e2lo, double e2hi,
                              cufftDoubleComplex *__restrict__ kern)
{
    const int j = j0 + (int)blockIdx.y;
    if (j >= nlm) return;
    int l = 0;
    while ((l + 1) * (l + 2) / 2 <= j) ++l;
    const int m = j - l * (l + 1) / 2;
    const size_t ncell = (size_t)G * G * G;
    kern += (size_t)blockIdx.y * ncell;
    const size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int iz = (int)(c % G), iy = (int)((c / G) % G), ix = (int)(c / ((size_t)G * G));
    const int half = G / 2;
    const int ox = (ix + half) % G - half, oy = (iy + half) % G - half, oz = (iz + half) % G - half; // numpy's (i + G/2) % G - G/2
    const double dx = h * ox, dy = h * oy, dz = h * oz;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    cufftDoubleComplex v = make_cuDoubleComplex(0.0, 0.0);
    if (r2 > 0.0 && r2 >= e2lo && r2 < e2hi) {
        const double rinv = rsqrt(r2);
        const double x = dx * rinv, y = dy * rinv, z = dz * rinv;
        double cr = 1.0, ci = 0.0; // (x + i y)^m
        for (int k = 0; k < m; ++k) { const double t = cr * x - ci * y; ci = cr * y + ci * x; cr = t; }
        const int comp = m == 0 ? l * l : l * l + 2 * m - 1;
        const double *yc = ycoef + (size_t)comp * (lmax + 1);
        double p = 0.0, zp = 1.0;
        for (int k = 0; k <= l - m; ++k) { p = fma(yc[k], zp, p); zp *= z; }
        v = make_cuDoubleComplex(p * cr, -p * ci); // conj(Y_lm)
    }
    kern[c] = v;
}

// kern[k] = fd[k] * conj(kern[k])   (cross-correlation in Fourier space)
__global__ void k_mesh_mul(const cufftDoubleComplex *__restrict__ fd, cufftDoubleComplex *__restrict__ kern, size_t ncell)
{
    const size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    kern += (size_t)blockIdx.y * ncell;
    const cufftDoubleComplex a = fd[c], b = kern[c];
    kern[c] = make_cuDoubleComplex(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// a_lm tile layout: alm[((g * ncomp + comp) * nb + b) * 32 + lane], cell = 32 g + lane
__global__ void k_mesh_scatter(const cufftDoubleComplex *__restrict__ field, size_t ncell, size_t npad, double scale, int ncomp, int nb,
                               int b, int j0, int nlm, double *__restrict__ alm)
{
    const size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    const int j = j0 + (int)blockIdx.y;
    if (c >= npad || j >= nlm) return;
    int l = 0;
    while ((l + 1) * (l + 2) / 2 <= j) ++l;
    const int m = j - l * (l + 1) / 2;
    const int cre = m == 0 ? l * l : l * l + 2 * m - 1, cim = m == 0 ? -1 : l * l + 2 * m;
    field += (size_t)blockIdx.y * ncell;
    const size_t g = c >> 5, lane = c & 31;
    const double re = c < ncell ? field[c].x * scale : 0.0, im = c < ncell ? field[c].y * scale : 0.0;
    alm[((g * ncomp + cre) * nb + b) * 32 + lane] = re;
    if (cim >= 0) alm[((g * ncomp + cim) * nb + b) * 32 + lane] = im;
}

} // namespace

// fd: G^3 complex scratch; kern: batch x G^3 complex scratch; alm: [npad/32][ncomp][nb][32]; gweights: [npad];
// plan1: cufftHandle for one G^3 Z2Z, planb: for `batch` of them (contiguous fields), both on stream s.  Per bin the
// (l, m >= 0) fields go through the FFTs `batch` at a time: 5 launches per batch instead of per field (a 64^3 mesh is
// launch-bound otherwise: 1050 launches for 10 bins, lmax = 5).
cudaError_t launch_mesh_alm(const double *delta, int G, double box, int lmax, int nb, const double *e2, const double *vinv,
                            const double *ycoef_dev, void *fd_, void *kern_, double *alm, double *gweights, int fft_plan1, int fft_planb,
                            int batch, cudaStream_t s, int *launches, int *fft_error)
{
    cufftDoubleComplex *fd = static_cast<cufftDoubleComplex *>(fd_), *kern = static_cast<cufftDoubleComplex *>(kern_);
    const size_t ncell = (size_t)G * G * G, npad = (ncell + 31) / 32 * 32;
    const double h = box / G, h3 = h * h * h;
    const int ncomp = (lmax + 1) * (lmax + 1), nlm = (lmax + 1) * (lmax + 2) / 2;
    const unsigned blocks = (unsigned)((npad + kT - 1) / kT);
    *fft_error = 0;
    k_mesh_weights<<<blocks, kT, 0, s>>>(delta, ncell, h3, fd, gweights, npad);
    *launches += 1;
    if (cufftExecZ2Z((cufftHandle)fft_plan1, fd, fd, CUFFT_FORWARD) != CUFFT_SUCCESS) { *fft_error = 1; return cudaSuccess; }
    cufftHandle planb = (cufftHandle)fft_planb;
    for (int b = 0; b < nb; ++b)
        for (int j0 = 0; j0 < nlm; j0 += batch) {
            // (a last, partial batch transforms the stale fields behind it as well; they are not read)
            const dim3 grid(blocks, (unsigned)batch);
            k_mesh_kernel<<<grid, kT, 0, s>>>(G, h, j0, nlm, lmax, ycoef_dev, e2[b], e2[b + 1], kern);
            if (cufftExecZ2Z(planb, kern, kern, CUFFT_FORWARD) != CUFFT_SUCCESS) { *fft_error = 1; return cudaSuccess; }
            k_mesh_mul<<<grid, kT, 0, s>>>(fd, kern, ncell);
            if (cufftExecZ2Z(planb, kern, kern, CUFFT_INVERSE) != CUFFT_SUCCESS) { *fft_error = 1; return cudaSuccess; }
            k_mesh_scatter<<<grid, kT, 0, s>>>(kern, ncell, npad, vinv[b] / (double)ncell, ncomp, nb, b, j0, nlm, alm);
            *launches += 3;
        }
    return cudaGetLastError();
}

int mesh_fft_plan_create(int G, int batch, cudaStream_t s, int *plan_out)
{
    cufftHandle p;
    int n[3] = {G, G, G};
    if (cufftPlanMany(&p, 3, n, nullptr, 1, G * G * G, nullptr, 1, G * G * G, CUFFT_Z2Z, batch) != CUFFT_SUCCESS) return 1;
    if (cufftSetStream(p, s) != CUFFT_SUCCESS) { cufftDestroy(p); return 1; }
    *plan_out = (int)p;
    return 0;
}

int mesh_fft_plan_set_stream(int plan, cudaStream_t s) { return cufftSetStream((cufftHandle)plan, s) == CUFFT_SUCCESS ? 0 : 1; }
void mesh_fft_plan_destroy(int plan) { cufftDestroy((cufftHandle)plan); }
