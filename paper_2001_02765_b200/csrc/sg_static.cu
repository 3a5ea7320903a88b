// sg_static.cu -- sg_force_uniform_static (include/sg_disk_static.h): the zeroth-order force sum on one uniform grid
// for callers that cannot let a library allocate device memory (an application arena that owns the whole GPU, a
// time-step loop that must not take cudaMalloc's device-wide synchronisation, a plug-in under a "no allocation"
// rule).  Self-contained on purpose: it shares no state with the context API of sg_api.cu.
//
// Mathematics as in sg_kernels.cu: regrouped by vertex, F^x_t = G sum_v w_v P(u_v, v_v) with
//   P(u, v) = -ln(v + r) = -s(v) ln(|v| + r) - [v < 0] 2 ln|u| ,     u = X_v - x_t, v = Y_v - y_t, r = sqrt(u^2 + v^2)
// hence F^x_t = -G (M^x + 2 S^x), M^x = sum_v w_v s(v) ln(|v| + r), S^x = sum_columns ln|u| * (weight below y_t),
// and x <-> y for F^y.  Lattice unit = half a cell: cell centres are odd, vertices even, so u and v are odd integers
// (never 0: no coincidence case on a uniform grid) and ln|u| comes from a table of ln(1), ln(3), ln(5), ...
//
// The vertex weights are the only data between the two kernels.  They live in g_static_w below, not in cudaMalloc'ed
// memory.
#include "../../include/sg_disk.h"
#include "../../include/sg_disk_static.h"

#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

#include <cuda_runtime.h>

namespace {

// The work array: part of the library image on every GPU that loads it, held until the process exits.
// In HOST code the name g_static_w is only a handle for cudaGetSymbolAddress -- it is not a device address and must
// never be passed to a kernel; scratch_address() below turns it into one, per device.
static __device__ __align__(256) double g_static_w[SG_STATIC_MAX_VERTICES];

constexpr int kStaticThreads = 128;
constexpr int kMaxDevices = 64;

std::mutex g_mu;
double *g_w_addr[kMaxDevices];          // device address of g_static_w on device d, nullptr until looked up
thread_local std::string g_err;

// Device address of g_static_w on `device`, which must be the CURRENT device (a __device__ variable has one
// instance per device and the look-up answers for the current one).  Looked up once per device, then cached.
cudaError_t scratch_address(int device, double **out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_w_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_w);
        if (e != cudaSuccess) return e;
        g_w_addr[device] = static_cast<double *>(p);
    }
    *out = g_w_addr[device];
    return cudaSuccess;
}

struct CurrentDevice {                  // work on `device`, give the caller's current device back
    int prev = -1;
    cudaError_t err;
    explicit CurrentDevice(int device) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        err = cudaSetDevice(device);
    }
    ~CurrentDevice() { if (prev >= 0) cudaSetDevice(prev); }
};

// w[a][b] (column a = 0..nx, b = 0..ny fastest) = signed sum of the <= 4 cells that have vertex (a, b) as a corner:
// + sigma where it is the cell's NE or SW corner, - sigma where NW or SE (the corner signs of [[.]]).
// Every entry the force kernel reads is written here first, so the array needs no clearing between calls.
__global__ void static_vertex_weights_kernel(const double *__restrict__ sigma, int nx, int ny, double *__restrict__ w) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (nx + 1) * (ny + 1)) return;
    const int a = idx / (ny + 1), b = idx - a * (ny + 1);
    const bool left = a > 0, right = a < nx, down = b > 0, up = b < ny;
    const double ne = (left && down) ? sigma[int64_t(b - 1) * nx + (a - 1)] : 0.0;   // v is that cell's NE corner
    const double nw = (right && down) ? sigma[int64_t(b - 1) * nx + a] : 0.0;        // ... NW corner
    const double se = (left && up) ? sigma[int64_t(b) * nx + (a - 1)] : 0.0;         // ... SE corner
    const double sw = (right && up) ? sigma[int64_t(b) * nx + a] : 0.0;              // ... SW corner
    w[idx] = ((ne - nw) - se) + sw;
}

// One target per thread, all vertices column by column (u, u^2 and ln|u| once per column); the weight of a vertex
// is the same address for the whole warp (one broadcast load).  Fixed order of summation: bit-reproducible.
__global__ void __launch_bounds__(kStaticThreads)
static_uniform_force_kernel(const double *__restrict__ w, int nx, int ny, double G, double *__restrict__ Fx,
                            double *__restrict__ Fy) {
    __shared__ double s_lnodd[SG_STATIC_MAX_SIDE];          // ln(2k + 1)
    const int m = max(nx, ny);
    for (int k = threadIdx.x; k < m; k += kStaticThreads) s_lnodd[k] = log(double(2 * k + 1));
    __syncthreads();

    const int n = nx * ny;
    const int t = blockIdx.x * kStaticThreads + threadIdx.x;
    const int tc = min(t, n - 1);                           // tail threads shadow the last target (warp stays converged)
    const int j = tc / nx, i = tc - j * nx;
    double Mx = 0.0, Sx = 0.0, My = 0.0, Sy = 0.0;
    for (int a = 0; a <= nx; ++a) {
        const int du = 2 * (a - i) - 1;
        const double u = double(du), au = fabs(u), uu = u * u;
        const double *__restrict__ wc = w + int64_t(a) * (ny + 1);
        double colM = 0.0, colB = 0.0, colY = 0.0, colS = 0.0;
        for (int b = 0; b <= ny; ++b) {
            const double wv = wc[b];
            const int dv = 2 * (b - j) - 1;
            const double v = double(dv), av = fabs(v);
            const double r = sqrt(fma(v, v, uu));           // exact integer under the root
            const double l1 = log(av + r), l2 = log(au + r);
            colM = fma(wv, dv < 0 ? -l1 : l1, colM);        // w s(v) ln(|v| + r)
            colB += dv < 0 ? wv : 0.0;                      // weight of this column below the target
            colY = fma(wv, l2, colY);                       // w ln(|u| + r); s(u) applied per column
            colS = fma(wv, s_lnodd[(abs(dv) - 1) >> 1], colS);   // w ln|v|, counted if the column is left of the target
        }
        Mx += colM;
        Sx = fma(s_lnodd[(abs(du) - 1) >> 1], colB, Sx);
        if (du < 0) { My -= colY; Sy += colS; } else { My += colY; }
    }
    if (t < n) {
        Fx[t] = -G * (Mx + 2.0 * Sx);
        Fy[t] = -G * (My + 2.0 * Sy);
    }
}

int fail(int code, const std::string &msg) {
    g_err = "sg_force_uniform_static: " + msg;
    return code;
}

}  // namespace

extern "C" {

int sg_force_uniform_static(int nx, int ny, double G, const double *sigma_dev, double *Fx_dev, double *Fy_dev,
                            int device, void *cuda_stream) {
    if (!sigma_dev || !Fx_dev || !Fy_dev) return fail(SG_ERR_ARG, "sigma_dev, Fx_dev and Fy_dev must not be NULL");
    if (!std::isfinite(G)) return fail(SG_ERR_ARG, "G must be finite");
    if (nx < 1 || ny < 1) return fail(SG_ERR_ARG, "nx and ny must be at least 1");
    if (nx > SG_STATIC_MAX_SIDE || ny > SG_STATIC_MAX_SIDE)
        return fail(SG_ERR_ARG, "grid side " + std::to_string(nx > ny ? nx : ny) + " exceeds SG_STATIC_MAX_SIDE = " +
                                    std::to_string(SG_STATIC_MAX_SIDE) + "; use sg_create / sg_force");
    const int64_t nv = int64_t(nx + 1) * (ny + 1);
    if (nv > SG_STATIC_MAX_VERTICES)
        return fail(SG_ERR_ARG, std::to_string(nx) + " x " + std::to_string(ny) + " cells need " + std::to_string(nv) +
                                    " vertex weights, the static work array holds SG_STATIC_MAX_VERTICES = " +
                                    std::to_string(SG_STATIC_MAX_VERTICES) + " (256 x 256 cells); use sg_create / sg_force");
    if (device < 0 || device >= kMaxDevices) return fail(SG_ERR_ARG, "device ordinal out of range");

    CurrentDevice cur(device);
    if (cur.err != cudaSuccess) return fail(SG_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(cur.err));
    double *w = nullptr;                // the DEVICE address of g_static_w on this device
    cudaError_t e = scratch_address(device, &w);
    if (e != cudaSuccess) return fail(SG_ERR_CUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));

    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    static_vertex_weights_kernel<<<unsigned((nv + 255) / 256), 256, 0, s>>>(sigma_dev, nx, ny, w);
    const int n = nx * ny;
    static_uniform_force_kernel<<<unsigned((n + kStaticThreads - 1) / kStaticThreads), kStaticThreads, 0, s>>>(
        w, nx, ny, G, Fx_dev, Fy_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SG_ERR_CUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
    return SG_OK;
}

const char *sg_static_last_error(void) { return g_err.c_str(); }

}  // extern "C"
