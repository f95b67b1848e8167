// moments_static.cu -- fp_cell_moments_static: the moment gather (a3, reading R0) for
// callers that may not allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  It needs no fp_ctx and calls no cudaMalloc / cudaFree / allocating library routine, ever.
//
// The kernels are the slice kernels of moments_seg.cuh (one-pass raw sums about a per-cell pivot in fp32x2, fp64 across
// lanes and slices, fp64 shift to central moments), which fp_cell_moments uses for few huge cells; they are correct for
// any cell sizes, and the only scratch they need is 28 fp64 accumulators per cell.  Here that scratch is a file-scope
// __device__ array of FP_STATIC_MAX_CELLS x 28 doubles (+ one status word): 3.5 MiB that every GPU which loads the
// library holds until the process exits.  The header is included a second time inside an anonymous namespace, so this
// translation unit has its own copies of the kernels and no existing code path changes.
//
// In host code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device with that device current (fps_setup).  Every call shares the array and
// it keeps the last call's contents: each call clears the accumulators and the status word it uses on its own stream
// before the kernels run; calls that overlap on the GPU (two streams, two threads) race on it.
#include "common.cuh"
#include "tiles.cuh"

#include <mutex>

namespace {
#include "moments_seg.cuh"
}

#define FPS_ACC_DOUBLES ((size_t)FP_STATIC_MAX_CELLS * 28)
#define FPS_TAIL_DOUBLES 32                                   // 256 B: the status word lives in the first 4 bytes

static __device__ __align__(256) double fps_scratch[FPS_ACC_DOUBLES + FPS_TAIL_DOUBLES];

#define FPS_MAX_DEVICES 64
static std::mutex fps_mutex;
static double* fps_ptr[FPS_MAX_DEVICES];                      // device address of fps_scratch, per device
static int fps_sms[FPS_MAX_DEVICES];
static thread_local char fps_err[256] = "";

static int fps_fail(int code, const char* msg)
{
    snprintf(fps_err, sizeof(fps_err), "%s", msg);
    return code;
}

extern "C" const char* fp_static_last_error(void) { return fps_err; }

// once per device, with that device current: the device address of the scratch array and the SM count
static int fps_setup(double** ptr, int* sms)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fps_fail(FP_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= FPS_MAX_DEVICES) return fps_fail(FP_ERR_UNSUPPORTED, "fp_cell_moments_static: device ordinal >= 64");
    std::lock_guard<std::mutex> lock(fps_mutex);
    if (!fps_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, fps_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(fps_err, sizeof(fps_err), "fp_cell_moments_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
            return FP_ERR_CUDA;
        }
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n < 1) return fps_fail(FP_ERR_CUDA, "fp_cell_moments_static: cannot read the SM count");
        fps_sms[dev] = n;
        fps_ptr[dev] = p;
    }
    *ptr = fps_ptr[dev];
    *sms = fps_sms[dev];
    return FP_OK;
}

extern "C" int fp_cell_moments_static(int64_t np, const float* vx, const float* vy, const float* vz,
                                      const int32_t* cell_start, int32_t ncell, int32_t mode, double* mom,
                                      uint32_t* d_status, void* stream)
{
    fps_err[0] = 0;
    if (ncell < 1 || !cell_start || !mom) return fps_fail(FP_ERR_ARG, "fp_cell_moments_static: ncell < 1 or null cell_start / mom");
    if (ncell > FP_STATIC_MAX_CELLS) {
        snprintf(fps_err, sizeof(fps_err), "fp_cell_moments_static: ncell = %d exceeds FP_STATIC_MAX_CELLS = %d (the static scratch "
                 "holds 28 doubles per cell); use fp_cell_moments with a context", ncell, FP_STATIC_MAX_CELLS);
        return FP_ERR_ARG;
    }
    if (mode != 0 && mode != 1) return fps_fail(FP_ERR_ARG, "fp_cell_moments_static: bad mode");
    if (np < 0 || np >= ((int64_t)1 << 31)) return fps_fail(FP_ERR_ARG, "fp_cell_moments_static: np outside [0, 2^31)");
    if (np > 0 && (!vx || !vy || !vz)) return fps_fail(FP_ERR_ARG, "fp_cell_moments_static: null velocity array");
    if (np > 0 && ((((uintptr_t)vx) | ((uintptr_t)vy) | ((uintptr_t)vz)) & 15u) != 0)
        return fps_fail(FP_ERR_ARG, "fp_cell_moments_static: vx, vy, vz must be 16-byte aligned (bulk copies)");
    double* acc = nullptr;
    int sms = 0;
    const int rc = fps_setup(&acc, &sms);
    if (rc != FP_OK) return rc;
    uint32_t* status = reinterpret_cast<uint32_t*>(acc + FPS_ACC_DOUBLES);
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the previous call's sums and status: clear what this call uses
    cudaError_t e = cudaMemsetAsync(acc, 0, (size_t)ncell * 28 * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(status, 0, FPS_TAIL_DOUBLES * sizeof(double), st);
    if (e != cudaSuccess) return fps_fail(FP_ERR_CUDA, cudaGetErrorString(e));
    const int cblocks = fp_div_up((int64_t)ncell + 1, 256);
    fp_launch(fp_cs_check_kernel, cblocks < 2 * sms ? cblocks : 2 * sms, 256, 0, st, cell_start, ncell, np, status, status);
    if (np > 0) {
        const int64_t nslices = (np + MOM_SEG - 1) / MOM_SEG;
        const int64_t want = (nslices + MOM_SEG_WARPS - 1) / MOM_SEG_WARPS;
        const int64_t cap = (int64_t)sms * 8;
        fp_launch(mom_seg_kernel, (int)(want < cap ? want : cap), MOM_SEG_WARPS * 32, 0, st, vx, vy, vz, cell_start, ncell, np, acc,
                  (const uint32_t*)status);
    }
    if (mode == 1)
        fp_launch(mom_seg_finalize_kernel<true>, fp_div_up(ncell, 128), 128, 0, st, vx, vy, vz, cell_start, ncell, (const double*)acc,
                  mom, (const uint32_t*)status);
    else
        fp_launch(mom_seg_finalize_kernel<false>, fp_div_up(ncell, 128), 128, 0, st, vx, vy, vz, cell_start, ncell, (const double*)acc,
                  mom, (const uint32_t*)status);
    e = cudaGetLastError();
    if (e == cudaSuccess && d_status) e = cudaMemcpyAsync(d_status, status, sizeof(uint32_t), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fps_fail(FP_ERR_CUDA, cudaGetErrorString(e));
    return FP_OK;
}
