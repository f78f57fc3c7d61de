// common.cu -- error plumbing shared by the translation units of a library.  Compiled into libu1gf.so, and once more
// (with -DU1GF_MEASURE_LIB) into libu1gf_measure.so, the roofline probes of include/u1gf_measure.h: each library keeps
// its own thread-local error text.
#include "u1gf_internal.h"

namespace u1gf {

static thread_local char t_err[512] = "";
thread_local int t_launches = 0;

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
}

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

int check_device() {
    static thread_local int cached = 1;  // 1 = unknown
    if (cached != 1) {
        if (cached != U1GF_OK) set_error("no CUDA device of compute capability 10.x (there is no CPU fallback)");
        return cached;
    }
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n < 1) {
        cudaGetLastError();
        cached = U1GF_ENODEV;
        return fail(U1GF_ENODEV, "no CUDA device available (%s); there is no CPU fallback",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    }
    int dev = 0;
    cudaGetDevice(&dev);
    int major = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (major != 10) {
        cached = U1GF_ENODEV;
        return fail(U1GF_ENODEV, "device %d has compute capability %d.x; libu1gf is built for sm_100a only", dev, major);
    }
    cached = U1GF_OK;
    return U1GF_OK;
}

}  // namespace u1gf

using namespace u1gf;

extern "C" {

#ifdef U1GF_MEASURE_LIB
const char* u1gf_measure_last_error(void) { return t_err; }
#else
const char* u1gf_last_error(void) { return t_err; }
int u1gf_abi_version(void) { return 3; }
int32_t u1gf_last_launch_count(void) { return t_launches; }
#endif

}  // extern "C"

