// fd_apply_hamiltonian_expect_static (declared and documented in include/fdham.h): the fused
// H psi + band energies + norms call for callers that must not
// allocate device memory.
//
// fd_apply_hamiltonian_expect needs scratch in global memory besides its inputs and outputs: the
// per-warp partial sums that the second, small launch adds up in a fixed order.  There the caller
// brings that scratch.  Some callers cannot: code that runs inside somebody else's memory budget
// (a plug-in of a host application whose pool owns every byte of the device and which forbids
// cudaMalloc in plug-ins), code on a latency path where cudaMalloc / cudaFree would synchronise the
// whole device, and code that has handed the device to a caching allocator it cannot reach from C.
// For them the scratch lives here, in a file-scope __device__ array that is part of the library
// image: the driver places it when the library's code is loaded on a device and keeps it until the
// process exits, and no call of this entry point allocates or frees anything.
//
// The array's name means two different things.  In device code it is the array.  In host code it is
// only a handle the runtime can look up: its address there is a host address, and a kernel handed
// that address would fault (or, on a system where the GPU can reach host memory, quietly use the
// wrong bytes).  The host side therefore asks the runtime for the device address once per device,
// with that device current, and passes that pointer to the kernels.
#include <mutex>

#include "../../include/fdham.h"
#include "fd_internal.h"

// One array per device that loads the library, FD_STATIC_SCRATCH_BYTES long, held until exit.
// Shared by every call of the entry point on that device, and it keeps what the last call wrote.
static __device__ __align__(256) unsigned char fd_static_scratch[FD_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
void *g_scratch_dev[kMaxDevices];  // device address of fd_static_scratch per device ordinal, or NULL

// Device address of the scratch array on `device`, which must be the current device.  The first
// call per device does the lookup (cudaGetSymbolAddress makes the runtime load the library's code
// on that device if it has not yet, which is why it should happen before any stream capture);
// later calls read the cached pointer.
int scratch_address(int device, void **ptr_out)
{
    if (device < 0 || device >= kMaxDevices) return FD_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_dev[device]) {
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, fd_static_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return FD_ERR_CUDA;
        }
        g_scratch_dev[device] = ptr;
    }
    *ptr_out = g_scratch_dev[device];
    return FD_OK;
}

}  // namespace

extern "C" int fd_apply_hamiltonian_expect_static(const fd_plan *plan, const void *psi,
                                                  const double *v_eff, void *out, double *eps,
                                                  double *norm, int64_t nbands, void *cuda_stream)
{
    if (!plan || nbands < 0) return FD_ERR_INVALID;
    // how much scratch this batch needs is a pure host computation on the plan
    const int64_t need = fd_expect_workspace_bytes(plan, nbands);
    if (need < 0) return (int)need;  // e.g. FD_ERR_UNSUPPORTED for single-precision plans
    if (need > (int64_t)FD_STATIC_SCRATCH_BYTES) return FD_ERR_SCRATCH;
    if (nbands == 0) return FD_OK;
    // the plan's device must be current: the lookup below and the launches go to the current device
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) {
        cudaGetLastError();
        return FD_ERR_CUDA;
    }
    if (cur != plan->device) return FD_ERR_INVALID;
    void *scratch = nullptr;
    const int rc = scratch_address(cur, &scratch);
    if (rc != FD_OK) return rc;
    // Nothing in the array has to start at zero: the kernels store every partial sum the reduction
    // launch of the same call reads (plain stores, no accumulation into the scratch), so what an
    // earlier call left behind is never read.  From here on this is the caller-workspace path with
    // the library's own array as the workspace: same kernels, same order of additions, same bits.
    return fd_apply_hamiltonian_expect(plan, psi, v_eff, out, eps, norm, nbands, scratch,
                                       (int64_t)FD_STATIC_SCRATCH_BYTES, cuda_stream);
}
