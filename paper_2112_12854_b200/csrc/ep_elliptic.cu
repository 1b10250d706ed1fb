// ep_elliptic.cu -- device-resident restarted GMRES for the elliptic equation of the bidomain model.
//
// "once v(t^{n+1}) is solved, the external potential v_ext(t^{n+1}) is obtained by solving the linear system
// given by the second equation of the system (6) through an iterative GMRES method with restart, using the external potential
// computed at previous time as first estimate".  PAPER.md:244 names the paper's own bottleneck: "the Arnoldi iteration and
// the solution of the corresponding Hessenberg system ... are based on the Lapack library running on the CPU".  Here the
// whole cycle stays on the device: the Krylov basis, the Hessenberg column, the Givens rotations and the triangular solve
// live in device memory and are advanced by kernels on the sim's stream; the host reads back one number (the residual
// estimate) every few iterations to decide when to stop.
//
// Orthogonalisation: classical Gram-Schmidt applied twice (one fused multi-dot launch + one fused update launch per pass
// instead of j+1 dot/axpy pairs), deterministic fixed-tree reductions.  No preconditioner (the paper names none).
#include "ep_kernels.cuh"

#include <algorithm>
#include <cmath>

namespace epk {

namespace {

constexpr int NB = 1024;   // partial-sum blocks of every reduction

// partial[q * NB + bx] = sum over this block's grid-stride of w[i] * V_q[i], q = 4 * blockIdx.y .. + 3 (< k)
__global__ void __launch_bounds__(256) multi_dot_partial_kernel(int64_t n, const double* __restrict__ w,
                                                                 const double* __restrict__ V, int64_t stride, int k,
                                                                 double* __restrict__ partial) {
    __shared__ double sh[4][256];
    const int q0 = 4 * blockIdx.y;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (k < 0) {            // plain sum of w into slot 0
        for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)NB * 256) acc[0] += w[i];
        k = 1;
    } else {
        for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)NB * 256) {
            const double wi = w[i];
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (q0 + q < k) acc[q] = fma(wi, V[(int64_t)(q0 + q) * stride + i], acc[q]);
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] = acc[q];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) {
#pragma unroll
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x < 4 && q0 + (int)threadIdx.x < k) partial[(int64_t)(q0 + threadIdx.x) * NB + blockIdx.x] = sh[threadIdx.x][0];
}

// out[q] (+)= sum_b partial[q * NB + b], fixed tree
__global__ void __launch_bounds__(256) multi_dot_final_kernel(const double* __restrict__ partial, double* __restrict__ out,
                                                               int accumulate) {
    __shared__ double sh[256];
    const double* p = partial + (int64_t)blockIdx.x * NB;
    sh[threadIdx.x] = (p[threadIdx.x] + p[threadIdx.x + 256]) + (p[threadIdx.x + 512] + p[threadIdx.x + 768]);
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[blockIdx.x] = accumulate ? out[blockIdx.x] + sh[0] : sh[0];
}

// w[i] += sign * sum_q coef[q] * V_q[i]
__global__ void __launch_bounds__(256) multi_axpy_kernel(int64_t n, double* __restrict__ w, const double* __restrict__ V,
                                                         int64_t stride, int k, const double* __restrict__ coef, double sign) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    double acc = 0.0;
    for (int q = 0; q < k; ++q) acc = fma(coef[q], V[(int64_t)q * stride + i], acc);
    w[i] = fma(sign, acc, w[i]);
}

// dst = b - Ax  (r0 of a cycle)
__global__ void __launch_bounds__(256) residual_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ Ax,
                                                       double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i < n) dst[i] = b[i] - Ax[i];
}

// dst = w / sqrt(norm2), or 0 on a (happy) breakdown
__global__ void __launch_bounds__(256) normalise_kernel(int64_t n, const double* __restrict__ w, const double* __restrict__ norm2,
                                                        double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const double s = norm2[0];
    dst[i] = s > 0.0 ? w[i] / sqrt(s) : 0.0;
}

// start of a cycle: g = (beta, 0, ..., 0), res = beta
__global__ void cycle_init_kernel(int m, const double* __restrict__ norm2, double* __restrict__ g, double* __restrict__ res) {
    const double beta = sqrt(norm2[0]);
    g[0] = beta;
    for (int i = 1; i <= m; ++i) g[i] = 0.0;
    res[0] = beta;
}

// column j of the Hessenberg matrix: previous rotations, the new one, the residual estimate |g_{j+1}|
__global__ void givens_kernel(int j, int m, const double* __restrict__ hcol, const double* __restrict__ norm2,
                              double* __restrict__ H, double* __restrict__ cs, double* __restrict__ sn,
                              double* __restrict__ g, double* __restrict__ res) {
    double* h = H + (int64_t)j * (m + 1);
    for (int i = 0; i <= j; ++i) h[i] = hcol[i];
    h[j + 1] = sqrt(norm2[0]);
    for (int i = 0; i < j; ++i) {
        const double t = cs[i] * h[i] + sn[i] * h[i + 1];
        h[i + 1] = -sn[i] * h[i] + cs[i] * h[i + 1];
        h[i] = t;
    }
    const double r = hypot(h[j], h[j + 1]);
    const double c = r > 0.0 ? h[j] / r : 1.0, s = r > 0.0 ? h[j + 1] / r : 0.0;
    cs[j] = c; sn[j] = s;
    h[j] = r; h[j + 1] = 0.0;
    g[j + 1] = -s * g[j];
    g[j] = c * g[j];
    res[0] = fabs(g[j + 1]);
}

// y = R^{-1} g for the first k columns
__global__ void back_substitute_kernel(int k, int m, const double* __restrict__ H, const double* __restrict__ g,
                                       double* __restrict__ y) {
    for (int i = k - 1; i >= 0; --i) {
        double acc = g[i];
        for (int c = i + 1; c < k; ++c) acc -= H[(int64_t)c * (m + 1) + i] * y[c];
        const double d = H[(int64_t)i * (m + 1) + i];
        y[i] = d != 0.0 ? acc / d : 0.0;
    }
}

__global__ void small_add_kernel(int k, double* __restrict__ a, const double* __restrict__ b) {
    const int i = threadIdx.x;
    if (i < k) a[i] += b[i];
}

// x[i] -= mean, mean = wsum / total (gauge: zero volume-weighted mean, reading E1)
__global__ void __launch_bounds__(256) shift_kernel(int64_t n, double* __restrict__ x, const double* __restrict__ wsum,
                                                    double inv_total) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i < n) x[i] -= wsum[0] * inv_total;
}

// first estimate by linear extrapolation in time: x <- 2 x - x_prev, x_prev <- x (the old one)
__global__ void __launch_bounds__(256) extrapolate_kernel(int64_t n, double* __restrict__ x, double* __restrict__ xprev, int have) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const double xo = x[i];
    if (have) x[i] = fma(2.0, xo, -xprev[i]);
    xprev[i] = xo;
}

inline unsigned blocks256(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

int gmres_alloc(Gmres& G, int64_t n, int m) {
    if (m < 1 || m > 63) return -2;
    G.n = n; G.m = m;
    G.stride = (n + 127) / 128 * 128;
    const size_t vec = sizeof(double) * (size_t)G.stride;
    if (cudaMalloc((void**)&G.V, vec * (m + 1)) != cudaSuccess) return -1;
    if (cudaMalloc((void**)&G.w, vec) != cudaSuccess) return -1;
    if (cudaMalloc((void**)&G.small, sizeof(double) * (size_t)((m + 1) * m + 5 * (m + 1) + 8)) != cudaSuccess) return -1;
    if (cudaMalloc((void**)&G.partial, sizeof(double) * (size_t)NB * (m + 4)) != cudaSuccess) return -1;
    G.H = G.small;
    G.cs = G.H + (size_t)(m + 1) * m;
    G.sn = G.cs + (m + 1);
    G.g = G.sn + (m + 1);
    G.y = G.g + (m + 1);
    G.hcol = G.y + (m + 1);
    G.scal = G.hcol + (m + 1);      // [0] norm^2, [1] residual estimate, [2] weighted sum
    G.bytes = (int64_t)(vec * (m + 2) + sizeof(double) * ((m + 1) * m + 5 * (m + 1) + 8) + sizeof(double) * NB * (m + 4));
    return 0;
}

void gmres_free(Gmres& G) {
    if (G.V) cudaFree(G.V);
    if (G.w) cudaFree(G.w);
    if (G.small) cudaFree(G.small);
    if (G.partial) cudaFree(G.partial);
    G = Gmres();
}

static void norm2_into(const Gmres& G, const double* x, double* out, cudaStream_t s) {
    multi_dot_partial_kernel<<<dim3(NB, 1), 256, 0, s>>>(G.n, x, x, G.stride, 1, G.partial);
    multi_dot_final_kernel<<<1, 256, 0, s>>>(G.partial, out, 0);
}

// Solves A x = b (A through `apply`), x holds the first estimate.  Returns iterations used (>= 0) or a negative CUDA error.
int gmres_solve(Gmres& G, const GmresOp& apply, const double* b, double* x, double rel_tol, double abs_tol, int max_cycles,
                int check_every, cudaStream_t s, double* rel_res_out, int64_t* launches) {
    const int m = G.m;
    const int64_t n = G.n;
    const unsigned gb = blocks256(n);
    double bnorm2 = 0.0;
    norm2_into(G, b, G.scal, s);
    *launches += 2;
    if (cudaMemcpyAsync(&bnorm2, G.scal, sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return -1;
    if (cudaStreamSynchronize(s) != cudaSuccess) return -1;
    const double bnorm = std::sqrt(bnorm2);
    if (!(bnorm > 0.0)) {                      // A x = 0 under the gauge: x = 0
        cudaMemsetAsync(x, 0, sizeof(double) * (size_t)n, s);
        if (rel_res_out) *rel_res_out = 0.0;
        return 0;
    }
    const double tol = std::max(rel_tol * bnorm, abs_tol);
    int iters = 0;
    double res = 0.0;
    for (int cycle = 0; cycle < max_cycles; ++cycle) {
        apply(x, G.w, s);                                                       // w = A x
        residual_kernel<<<gb, 256, 0, s>>>(n, b, G.w, G.w);                     // w = b - A x
        norm2_into(G, G.w, G.scal, s);
        cycle_init_kernel<<<1, 1, 0, s>>>(m, G.scal, G.g, G.scal + 1);
        normalise_kernel<<<gb, 256, 0, s>>>(n, G.w, G.scal, G.V);               // v_0
        *launches += apply.launches + 5;
        if (cudaMemcpyAsync(&res, G.scal + 1, sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return -1;
        if (cudaStreamSynchronize(s) != cudaSuccess) return -1;
        if (res <= tol) break;
        int k = 0;                                                              // columns built in this cycle
        for (int j = 0; j < m; ++j) {
            const double* vj = G.V + (size_t)j * G.stride;
            apply(vj, G.w, s);                                                  // w = A v_j
            const int kk = j + 1;
            const dim3 grid(NB, (unsigned)((kk + 3) / 4));
            for (int pass = 0; pass < 2; ++pass) {                              // classical Gram-Schmidt, twice
                multi_dot_partial_kernel<<<grid, 256, 0, s>>>(n, G.w, G.V, G.stride, kk, G.partial);
                multi_dot_final_kernel<<<kk, 256, 0, s>>>(G.partial, pass == 0 ? G.hcol : G.y, 0);
                multi_axpy_kernel<<<gb, 256, 0, s>>>(n, G.w, G.V, G.stride, kk, pass == 0 ? G.hcol : G.y, -1.0);
                if (pass == 1) small_add_kernel<<<1, 64, 0, s>>>(kk, G.hcol, G.y);                            // hcol += second-pass dots
            }
            norm2_into(G, G.w, G.scal, s);
            givens_kernel<<<1, 1, 0, s>>>(j, m, G.hcol, G.scal, G.H, G.cs, G.sn, G.g, G.scal + 1);
            normalise_kernel<<<gb, 256, 0, s>>>(n, G.w, G.scal, G.V + (size_t)(j + 1) * G.stride);
            *launches += apply.launches + 11;
            ++iters; k = j + 1;
            if ((j + 1) % check_every == 0 || j + 1 == m) {
                if (cudaMemcpyAsync(&res, G.scal + 1, sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return -1;
                if (cudaStreamSynchronize(s) != cudaSuccess) return -1;
                if (res <= tol) break;
            }
        }
        back_substitute_kernel<<<1, 1, 0, s>>>(k, m, G.H, G.g, G.y);
        multi_axpy_kernel<<<gb, 256, 0, s>>>(n, x, G.V, G.stride, k, G.y, 1.0);  // x += V_k y
        *launches += 2;
        if (res <= tol) break;
    }
    if (rel_res_out) *rel_res_out = res <= abs_tol ? std::min(res / bnorm, rel_tol) : res / bnorm;
    if (cudaGetLastError() != cudaSuccess) return -1;
    return iters;
}

// x -= (sum_i x[i]) / n: makes a right-hand side compatible with an operator whose left null vector is the constant
void launch_remove_mean(const Gmres& G, double* x, cudaStream_t s) {
    multi_dot_partial_kernel<<<dim3(NB, 1), 256, 0, s>>>(G.n, x, nullptr, G.stride, -1, G.partial);
    multi_dot_final_kernel<<<1, 256, 0, s>>>(G.partial, G.scal + 2, 0);
    shift_kernel<<<blocks256(G.n), 256, 0, s>>>(G.n, x, G.scal + 2, 1.0 / (double)G.n);
}

void launch_extrapolate(int64_t n, double* x, double* xprev, int have, cudaStream_t s) {
    extrapolate_kernel<<<blocks256(n), 256, 0, s>>>(n, x, xprev, have);
}

void launch_remove_weighted_mean(const Gmres& G, double* x, const double* weight, double total, cudaStream_t s) {
    multi_dot_partial_kernel<<<dim3(NB, 1), 256, 0, s>>>(G.n, x, weight, G.stride, 1, G.partial);
    multi_dot_final_kernel<<<1, 256, 0, s>>>(G.partial, G.scal + 2, 0);
    shift_kernel<<<blocks256(G.n), 256, 0, s>>>(G.n, x, G.scal + 2, 1.0 / total);
}

}  // namespace epk
