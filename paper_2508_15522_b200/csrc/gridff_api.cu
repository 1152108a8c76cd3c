// gridff_api.cu — error reporting, counters and the small host-side helpers of the C-ABI (include/gridff.h).
#include "gridff_internal.cuh"
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <atomic>

namespace gridff {

static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches{0};

void set_error(const char* fmt, ...) {
    va_list ap; va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what) {
    set_error("CUDA error in %s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    cudaGetLastError();
    return GRIDFF_ECUDA;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

}  // namespace gridff

extern "C" {

const char* gridff_last_error(void) { return gridff::g_err; }

int gridff_version(void) { return 100; }

long long gridff_launch_count(void) { return gridff::g_launches.load(std::memory_order_relaxed); }

int gridff_atom_coefs(double alpha, int n, const float* e, const float* R, const float* q, float* coef) {
    if (n < 0 || (n > 0 && (!e || !R || !coef))) { gridff::set_error("bad arguments to gridff_atom_coefs"); return GRIDFF_EINVAL; }
    for (int i = 0; i < n; ++i) {
        // PAPER.md:L83-85 Eq. 4 with e_i = sqrt(eps_i): P_i = e_i exp(2 alpha R_i), L_i = -2 e_i exp(alpha R_i)
        coef[4 * i] = (float)((double)e[i] * exp(2.0 * alpha * (double)R[i]));
        coef[4 * i + 1] = (float)(-2.0 * (double)e[i] * exp(alpha * (double)R[i]));
        coef[4 * i + 2] = q ? q[i] : 0.0f;
        coef[4 * i + 3] = 0.0f;
    }
    return GRIDFF_OK;
}

}  // extern "C"
