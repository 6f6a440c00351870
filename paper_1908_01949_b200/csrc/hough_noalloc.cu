// cdc_hough_seed_ranges_noalloc: the A2 Hough vote (hough.cu, reading C13) for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The hits come as
// plain device arrays (no cdc_events handle, whose creation allocates) and the one piece of scratch the vote needs, the
// per-event packed peak key (votes << 32 | ~linear bin) that hough_vote_kernel reduces into with atomicMax and
// hough_finalize_kernel reads, lives in a file-scope device array of fixed size instead of in the events' slab.
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device
// with cudaGetSymbolAddress (here, in the file that defines it) and passed to the kernels as a pointer.
#include <mutex>

#include "cdc_internal.cuh"

namespace {

// 4096 events x 8 B = 32 KB of device memory on every GPU that loads the library, until exit
static __device__ __align__(256) unsigned long long g_hough_peak_key[CDC_HOUGH_NOALLOC_MAX_EVENTS];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned long long *g_key_ptr[kMaxDevices] = {};

// device address of the scratch on the CURRENT device (looked up once per device)
cudaError_t scratch_of_current_device(unsigned long long **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_key_ptr[dev]) {
        unsigned long long *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_hough_peak_key);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_key_ptr[dev] = p;
    }
    *out = g_key_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int32_t cdc_hough_seed_ranges_noalloc(const cdc_geometry *g, int32_t n_events, const int32_t *d_hit_offsets,
                                                 const int32_t *d_wire_id, const cdc_hough_params *hp, int32_t charge,
                                                 const float *d_zref_mm, double *d_ranges, int32_t *d_peak,
                                                 uint32_t *d_accum_or_null, void *stream)
{
    return cdc_guard("cdc_hough_seed_ranges_noalloc", [&]() -> int32_t {
    if (!g || !hp) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges_noalloc: null argument");
    if (n_events < 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges_noalloc: n_events < 0");
    if (n_events > CDC_HOUGH_NOALLOC_MAX_EVENTS)
        CDC_FAIL(CDC_ERR_RANGE, "cdc_hough_seed_ranges_noalloc: n_events exceeds CDC_HOUGH_NOALLOC_MAX_EVENTS (4096), the size of "
                                "the static scratch: split the batch, or use cdc_hough_seed_ranges");
    if (charge != 1 && charge != -1) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges_noalloc: charge must be +-1");
    int32_t dims[3];
    const int32_t rc = cdc_hough_dims(hp, dims);
    if (rc != CDC_OK) return rc;
    unsigned long long *d_key = nullptr;
    CDC_CUDA(scratch_of_current_device(&d_key));          // set-up: the first call on a device resolves the address
    if (n_events == 0) return CDC_OK;                     // (a call with no events is a set-up call: nothing is launched)
    if (!d_hit_offsets || !d_wire_id || !d_zref_mm || !d_ranges || !d_peak)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges_noalloc: null argument");
    HoughLaunch L;
    L.n_events = n_events; L.nR = dims[0]; L.ncy = dims[1]; L.ncx = dims[2];
    L.bin_xy = (float)hp->bin_xy_mm; L.bin_R = (float)hp->bin_R_mm; L.tol = (float)hp->tol_mm; L.R_lo = (float)hp->R_lo_mm;
    L.half_xy = (float)hp->half_xy_mm; L.origin = (float)hp->origin_mm;
    L.bin_xy64 = hp->bin_xy_mm; L.bin_R64 = hp->bin_R_mm; L.R_lo64 = hp->R_lo_mm; L.half_xy64 = hp->half_xy_mm;
    L.R0 = g->R0; L.half_theta = hp->half_theta_rad; L.half_pt = hp->half_pt_MeV; L.bz = g->field.bz_T; L.charge = charge;
    L.d_wire5 = g->d_wire5; L.d_offsets = d_hit_offsets; L.d_wire_id = d_wire_id; L.d_zref = d_zref_mm;
    L.d_ranges = d_ranges; L.d_peak = d_peak; L.d_accum = d_accum_or_null;
    L.d_peak_key = d_key;                                 // launch_hough clears the n_events keys it uses (cudaMemsetAsync on `stream`)
    CDC_CUDA(launch_hough(L, (cudaStream_t)stream));
    return CDC_OK;
    });
}
