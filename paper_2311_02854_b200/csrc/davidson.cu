// dmrg_davidson: single-root Davidson eigensolver around dmrg_sigma (Ref. 74).
// The paper keeps the subspace algebra on CPU rank 0 and ships the trial vector / sigma vector
// across PCIe and NCCL every iteration; here every vector lives in HBM, all
// O(n) work is done by the kernels below, and the host only sees the m x m subspace matrix.
// Reductions use a fixed grid and a fixed summation tree, so results are reproducible run to run.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <new>

#include "plan.h"

struct DavidsonWs {
    int64_t n = 0, stride = 0;   // stride: vector pitch (even, keeps every vector 16-byte aligned)
    int max_space = 0;
    double *B = nullptr, *W = nullptr;   // max_space vectors each
    double *x = nullptr, *r = nullptr, *hd = nullptr;
    double *partial = nullptr;           // [max_space+2][RED_GRID]
    double *scal = nullptr;              // device scalars: [0..max_space) dots, [max_space..) misc
    double *y = nullptr;                 // device copy of the Ritz coefficients
};

namespace dmrg {

constexpr int RED_GRID = 592;   // 4 CTAs per SM
constexpr int RED_BLOCK = 256;

void davidson_ws_free(DavidsonWs* ws) {
    if (!ws) return;
    cudaFree(ws->B); cudaFree(ws->W); cudaFree(ws->x); cudaFree(ws->r); cudaFree(ws->hd);
    cudaFree(ws->partial); cudaFree(ws->scal); cudaFree(ws->y);
    delete ws;
}

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[RED_BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < RED_BLOCK / 32; i++) s += sh[i];
    return s;   // valid on thread 0
}

// partial[i*RED_GRID + cta] = sum over this CTA's slice of V_i[e] * w[e]
__global__ void __launch_bounds__(RED_BLOCK) dots_partial_kernel(const double* __restrict__ V, int64_t stride, int m,
                                                                 const double* __restrict__ w, int64_t n, double* __restrict__ partial) {
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    const int64_t e0 = per * blockIdx.x, e1 = min(n, e0 + per);
    for (int i = 0; i < m; i++) {
        const double* v = V + (int64_t)i * stride;
        double acc = 0.0;
        for (int64_t e = e0 + threadIdx.x; e < e1; e += RED_BLOCK) acc = fma(v[e], w[e], acc);
        const double s = block_sum(acc);
        if (threadIdx.x == 0) partial[(int64_t)i * RED_GRID + blockIdx.x] = s;
    }
}
// out[i] = sum_cta partial[i][cta]  in cta order
__global__ void dots_final_kernel(const double* __restrict__ partial, int m, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    double s = 0.0;
    for (int c = 0; c < RED_GRID; c++) s += partial[(int64_t)i * RED_GRID + c];
    out[i] = s;
}

// x = sum_i y_i b_i ; r = sum_i y_i w_i - theta x
__global__ void __launch_bounds__(256) ritz_kernel(const double* __restrict__ B, const double* __restrict__ W, int64_t stride, int m,
                                                   const double* __restrict__ y, double theta, int64_t n,
                                                   double* __restrict__ x, double* __restrict__ r) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        double xs = 0.0, hs = 0.0;
        for (int i = 0; i < m; i++) {
            const double yi = y[i];
            xs = fma(yi, B[(int64_t)i * stride + e], xs);
            hs = fma(yi, W[(int64_t)i * stride + e], hs);
        }
        x[e] = xs;
        r[e] = hs - theta * xs;
    }
}
// t = r * den / (den^2 + delta^2), den = theta - hd   (in place on r)
__global__ void __launch_bounds__(256) precond_kernel(double* __restrict__ r, const double* __restrict__ hd, double theta, double delta, int64_t n) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const double den = theta - hd[e];
        r[e] = r[e] * den / (den * den + delta * delta);
    }
}
// t -= sum_i c_i b_i
__global__ void __launch_bounds__(256) project_out_kernel(double* __restrict__ t, const double* __restrict__ B, int64_t stride, int m,
                                                          const double* __restrict__ c, int64_t n) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int i = 0; i < m; i++) s = fma(c[i], B[(int64_t)i * stride + e], s);
        t[e] -= s;
    }
}
// dst = src / sqrt(*norm2)
__global__ void __launch_bounds__(256) normalize_kernel(double* __restrict__ dst, const double* __restrict__ src, const double* __restrict__ norm2, int64_t n) {
    const double s = 1.0 / sqrt(*norm2);
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) dst[e] = src[e] * s;
}

// cyclic Jacobi for a symmetric m x m matrix (row-major a, destroyed); returns lowest eigenpair
static void jacobi_lowest(std::vector<double>& a, int m, double* eval, std::vector<double>& evec) {
    std::vector<double> v((size_t)m * m, 0.0);
    for (int i = 0; i < m; i++) v[(size_t)i * m + i] = 1.0;
    for (int sweep = 0; sweep < 100; sweep++) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < m; i++) {
            diag += a[(size_t)i * m + i] * a[(size_t)i * m + i];
            for (int j = i + 1; j < m; j++) off += a[(size_t)i * m + j] * a[(size_t)i * m + j];
        }
        if (off <= 1e-32 * std::max(diag, 1e-300)) break;
        for (int p = 0; p < m; p++)
            for (int q = p + 1; q < m; q++) {
                const double apq = a[(size_t)p * m + q];
                if (apq == 0.0) continue;
                const double app = a[(size_t)p * m + p], aqq = a[(size_t)q * m + q];
                const double tau = (aqq - app) / (2.0 * apq);
                const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                for (int k = 0; k < m; k++) {
                    const double akp = a[(size_t)k * m + p], akq = a[(size_t)k * m + q];
                    a[(size_t)k * m + p] = c * akp - s * akq;
                    a[(size_t)k * m + q] = s * akp + c * akq;
                }
                for (int k = 0; k < m; k++) {
                    const double apk = a[(size_t)p * m + k], aqk = a[(size_t)q * m + k];
                    a[(size_t)p * m + k] = c * apk - s * aqk;
                    a[(size_t)q * m + k] = s * apk + c * aqk;
                }
                for (int k = 0; k < m; k++) {
                    const double vkp = v[(size_t)k * m + p], vkq = v[(size_t)k * m + q];
                    v[(size_t)k * m + p] = c * vkp - s * vkq;
                    v[(size_t)k * m + q] = s * vkp + c * vkq;
                }
            }
    }
    int lo = 0;
    for (int i = 1; i < m; i++)
        if (a[(size_t)i * m + i] < a[(size_t)lo * m + lo]) lo = i;
    *eval = a[(size_t)lo * m + lo];
    evec.resize(m);
    for (int k = 0; k < m; k++) evec[k] = v[(size_t)k * m + lo];
}

static int ws_ensure(dmrg_plan* P, int max_space) {
    const int64_t n = P->psi_size;
    if (P->dav && P->dav->max_space >= max_space) return DMRG_OK;
    if (P->dav) { davidson_ws_free(P->dav); P->dav = nullptr; }
    DavidsonWs* ws = new (std::nothrow) DavidsonWs();
    if (!ws) { set_error("dmrg_davidson: out of host memory"); return DMRG_ENOMEM; }
    ws->n = n; ws->stride = round_up2(n); ws->max_space = max_space;
    const size_t vb = sizeof(double) * (size_t)ws->stride;
    // the workspace is attached to the plan only once every allocation has succeeded
    auto alloc_all = [&]() -> int {
        DMRG_CUDA(cudaMalloc(&ws->B, vb * max_space));
        DMRG_CUDA(cudaMalloc(&ws->W, vb * max_space));
        DMRG_CUDA(cudaMalloc(&ws->x, vb));
        DMRG_CUDA(cudaMalloc(&ws->r, vb));
        DMRG_CUDA(cudaMalloc(&ws->hd, vb));
        DMRG_CUDA(cudaMalloc(&ws->partial, sizeof(double) * (size_t)(max_space + 2) * RED_GRID));
        DMRG_CUDA(cudaMalloc(&ws->scal, sizeof(double) * (size_t)(max_space + 8)));
        DMRG_CUDA(cudaMalloc(&ws->y, sizeof(double) * (size_t)(max_space + 8)));
        return DMRG_OK;
    };
    const int rc = alloc_all();
    if (rc != DMRG_OK) { davidson_ws_free(ws); return rc; }
    P->dav = ws;
    return DMRG_OK;
}

static int dots(DavidsonWs* ws, const double* V, int m, const double* w, double* out, cudaStream_t st) {
    dots_partial_kernel<<<RED_GRID, RED_BLOCK, 0, st>>>(V, ws->stride, m, w, ws->n, ws->partial);
    dots_final_kernel<<<(m + 63) / 64, 64, 0, st>>>(ws->partial, m, out);
    DMRG_CUDA(cudaGetLastError());
    return DMRG_OK;
}

static int davidson_impl(dmrg_plan* P, double* x_io, int max_iter, int max_space, double tol, double* energy,
                         double* resid_norm, int* iters, double* thetas, cudaStream_t st) {
    const double delta = 1e-3;
    int rc = ws_ensure(P, max_space);
    if (rc) return rc;
    DavidsonWs* ws = P->dav;
    const int64_t n = ws->n, ld = ws->stride;
    const int EW_GRID = 1184;
    double* s_dots = ws->scal;                 // [max_space]
    double* s_misc = ws->scal + max_space;     // [8]
    std::vector<double> G((size_t)max_space * max_space, 0.0), col(max_space + 8), yv;
    if ((rc = dmrg_hdiag(P, ws->hd, st))) return rc;
    // b_0 = x0 / |x0|
    if ((rc = dots(ws, x_io, 1, x_io, s_misc, st))) return rc;
    {
        double n2 = 0.0;
        DMRG_CUDA(cudaMemcpyAsync(&n2, s_misc, sizeof(double), cudaMemcpyDeviceToHost, st));
        DMRG_CUDA(cudaStreamSynchronize(st));
        if (!(n2 > 0.0) || !std::isfinite(n2)) { set_error("dmrg_davidson: the initial guess has norm^2 = %g", n2); return DMRG_EINVAL; }
    }
    normalize_kernel<<<EW_GRID, 256, 0, st>>>(ws->B, x_io, s_misc, n);
    int m = 1, it = 0;
    double theta = 0.0, rn = 0.0;
    bool have_x = false;
    while (it < max_iter) {
        double* bm = ws->B + (int64_t)(m - 1) * ld;
        double* wm = ws->W + (int64_t)(m - 1) * ld;
        if ((rc = dmrg_sigma(P, bm, wm, st))) return rc;
        it++;
        if ((rc = dots(ws, ws->B, m, wm, s_dots, st))) return rc;
        DMRG_CUDA(cudaMemcpyAsync(col.data(), s_dots, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
        DMRG_CUDA(cudaStreamSynchronize(st));
        for (int i = 0; i < m; i++) G[(size_t)i * max_space + (m - 1)] = G[(size_t)(m - 1) * max_space + i] = col[i];
        std::vector<double> a((size_t)m * m);
        for (int i = 0; i < m; i++)
            for (int j = 0; j < m; j++) a[(size_t)i * m + j] = G[(size_t)i * max_space + j];
        jacobi_lowest(a, m, &theta, yv);
        DMRG_CUDA(cudaMemcpyAsync(ws->y, yv.data(), sizeof(double) * m, cudaMemcpyHostToDevice, st));
        ritz_kernel<<<EW_GRID, 256, 0, st>>>(ws->B, ws->W, ld, m, ws->y, theta, n, ws->x, ws->r);
        have_x = true;
        if ((rc = dots(ws, ws->r, 1, ws->r, s_misc, st))) return rc;
        double rn2 = 0.0;
        DMRG_CUDA(cudaMemcpyAsync(&rn2, s_misc, sizeof(double), cudaMemcpyDeviceToHost, st));
        DMRG_CUDA(cudaStreamSynchronize(st));
        rn = std::sqrt(rn2);
        if (thetas) thetas[it - 1] = theta;
        if (rn <= tol || it >= max_iter) break;
        if (m >= max_space) {   // collapse to {x}
            if ((rc = dots(ws, ws->x, 1, ws->x, s_misc, st))) return rc;
            normalize_kernel<<<EW_GRID, 256, 0, st>>>(ws->B, ws->x, s_misc, n);
            std::fill(G.begin(), G.end(), 0.0);
            m = 1;
            continue;
        }
        precond_kernel<<<EW_GRID, 256, 0, st>>>(ws->r, ws->hd, theta, delta, n);
        for (int pass = 0; pass < 2; pass++) {   // classical Gram-Schmidt, twice
            if ((rc = dots(ws, ws->B, m, ws->r, s_dots, st))) return rc;
            project_out_kernel<<<EW_GRID, 256, 0, st>>>(ws->r, ws->B, ld, m, s_dots, n);
        }
        if ((rc = dots(ws, ws->r, 1, ws->r, s_misc, st))) return rc;
        {   // a correction vector that vanishes after orthogonalisation (exact eigenvector inside the space) cannot
            // extend the basis: report it instead of dividing by zero (rn > tol here, so this is a breakdown)
            double t2 = 0.0;
            DMRG_CUDA(cudaMemcpyAsync(&t2, s_misc, sizeof(double), cudaMemcpyDeviceToHost, st));
            DMRG_CUDA(cudaStreamSynchronize(st));
            if (!(t2 > 1e-300) || !std::isfinite(t2)) {
                set_error("dmrg_davidson: the new direction has norm^2 = %g after orthogonalisation (iteration %d)", t2, it);
                break;
            }
        }
        normalize_kernel<<<EW_GRID, 256, 0, st>>>(ws->B + (int64_t)m * ld, ws->r, s_misc, n);
        DMRG_CUDA(cudaGetLastError());
        m++;
    }
    if (have_x) {
        if ((rc = dots(ws, ws->x, 1, ws->x, s_misc, st))) return rc;
        normalize_kernel<<<EW_GRID, 256, 0, st>>>(x_io, ws->x, s_misc, n);
    }
    DMRG_CUDA(cudaGetLastError());
    DMRG_CUDA(cudaStreamSynchronize(st));
    if (energy) *energy = theta;
    if (resid_norm) *resid_norm = rn;
    if (iters) *iters = it;
    if (rn > tol) { set_error("dmrg_davidson: not converged after %d iterations (|r| = %.3e)", it, rn); return DMRG_ENOCONV; }
    return DMRG_OK;
}

}  // namespace dmrg

extern "C" int dmrg_davidson(dmrg_plan* plan, double* x, int32_t max_iter, int32_t max_space, double tol, double* energy,
                             double* resid_norm, int32_t* iters, double* thetas, void* cuda_stream) {
    if (!plan || !x || max_iter < 1) { dmrg::set_error("dmrg_davidson: bad argument"); return DMRG_EINVAL; }
    if (max_space < 2 && max_iter > 1) { dmrg::set_error("dmrg_davidson: max_space must be >= 2 (a space of one vector can never be extended)"); return DMRG_EINVAL; }
    if (max_space < 1) { dmrg::set_error("dmrg_davidson: max_space must be >= 1"); return DMRG_EINVAL; }
    if (plan->ops->structure_only) { dmrg::set_error("dmrg_davidson: the operator store was loaded without values (planning only)"); return DMRG_EINVAL; }
    if ((uintptr_t)x & 15) { dmrg::set_error("dmrg_davidson: x must be 16-byte aligned"); return DMRG_EINVAL; }
    try {
        return dmrg::davidson_impl(plan, x, max_iter, max_space, tol, energy, resid_norm, iters, thetas, (cudaStream_t)cuda_stream);
    } catch (const std::bad_alloc&) {
        dmrg::set_error("dmrg_davidson: out of host memory");
        return DMRG_ENOMEM;
    }
}

// ---------------------------------------------------------------------------------------------
// dmrg_dots_static: the Davidson dot-product pair (dots_partial_kernel + dots_final_kernel above) for callers that
// may not allocate: the per-CTA partial sums, which dmrg_davidson keeps in a cudaMalloc'ed workspace, live in a
// file-scope device array instead.  In HOST code `g_dots_scratch` is only a stand-in for the symbol, not a device
// address: the address is looked up once per device with cudaGetSymbolAddress and handed to the kernels.
namespace dmrg {

constexpr int DOTS_STATIC_MAX_VECTORS = DMRG_DOTS_STATIC_MAX_VECTORS;
constexpr int DOTS_STATIC_MAX_DEVICES = 64;
static __device__ __align__(256) double g_dots_scratch[(size_t)DOTS_STATIC_MAX_VECTORS * RED_GRID];   // 151552 bytes per GPU

static std::atomic<double*> g_dots_scratch_ptr[DOTS_STATIC_MAX_DEVICES];   // device address of g_dots_scratch per device ordinal (null = not looked up yet)

// Device address of the scratch array on the CURRENT device (looked up on first use there; idempotent, so two threads
// racing on the first call store the same pointer).  No allocation: the array is part of the loaded module.
static int dots_scratch_address(double** out) {
    int dev = -1;
    DMRG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= DOTS_STATIC_MAX_DEVICES) { set_error("dmrg_dots_static: device ordinal %d is outside [0, %d)", dev, DOTS_STATIC_MAX_DEVICES); return DMRG_EINVAL; }
    double* p = g_dots_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        DMRG_CUDA(cudaGetSymbolAddress((void**)&p, g_dots_scratch));
        if (!p) { set_error("dmrg_dots_static: cudaGetSymbolAddress returned a null address on device %d", dev); return DMRG_ECUDA; }
        g_dots_scratch_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return DMRG_OK;
}

}  // namespace dmrg

extern "C" int dmrg_dots_static(const double* V, int64_t stride, int32_t m, const double* w, int64_t n, double* out, void* cuda_stream) {
    using namespace dmrg;
    if (!V || !w || !out) { set_error("dmrg_dots_static: null pointer"); return DMRG_EINVAL; }
    if (m < 1 || m > DOTS_STATIC_MAX_VECTORS) {
        set_error("dmrg_dots_static: m = %d vectors is outside [1, %d] (the static scratch holds %d x %d partial sums; use dmrg_davidson's own workspace path for more)",
                  m, DOTS_STATIC_MAX_VECTORS, DOTS_STATIC_MAX_VECTORS, RED_GRID);
        return DMRG_EINVAL;
    }
    if (n < 0 || (m > 1 && stride < n)) { set_error("dmrg_dots_static: bad n = %lld / stride = %lld", (long long)n, (long long)stride); return DMRG_EINVAL; }
    double* scratch = nullptr;
    const int rc = dots_scratch_address(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // every partial sum dots_final_kernel reads (m rows x RED_GRID CTAs) is written by dots_partial_kernel in this very
    // call -- CTAs with an empty slice store 0 -- so nothing left behind by an earlier call is ever read and nothing needs clearing
    dots_partial_kernel<<<RED_GRID, RED_BLOCK, 0, st>>>(V, stride, m, w, n, scratch);
    dots_final_kernel<<<(m + 63) / 64, 64, 0, st>>>(scratch, m, out);
    DMRG_CUDA(cudaGetLastError());
    return DMRG_OK;
}
