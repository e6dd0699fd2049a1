// energy_static.cu -- tkhp_polar_energy_static: the polarization energy for callers that cannot
// allocate device memory (include/tkhp.h has the contract).
//
// Every other entry point of libtkhp works out of a context, and a context needs a workspace that
// somebody allocated with cudaMalloc, plus the streams, events and pinned buffers tkhp_create makes.
// Some users of the energy reduction have none of that to give: a force-field plug-in called from
// inside an MD engine's step loop after the engine has handed all device memory to its own pool; a
// callback that runs while another host thread has a stream capture open (cudaMalloc is refused
// then); a latency-bound integrator that cannot take the device-wide stall of cudaMalloc/cudaFree
// in the middle of a step.  They hold mu and the field on the device already and want E_pol.
//
// The reduction of k_energy (pcg.cu) needs one partial sum per CTA and a ticket counter in global
// memory.  Here that scratch is a fixed array in the library's own device image: it exists on every
// GPU that loads libtkhp, from module load until the process exits, and no call creates or frees it.
// Nothing in this file calls cudaMalloc, cudaFree, cudaHostAlloc or any routine that allocates.
//
// The arithmetic and its order are those of k_energy (same block size, same grid rule, same
// fixed-order re-reduction by the last CTA), so the result equals tkhp_polar_energy's for FP64 and
// MIXED contexts bit for bit.
#include <mutex>

#include "common.cuh"
#include "reduce.cuh"

namespace tkhp {

void set_thread_error(const char *msg);   // api.cu: the text tkhp_last_error(NULL) returns

// ---- the scratch -----------------------------------------------------------------------------
// Layout: STATIC_PARTIALS doubles (one per CTA), then one 256-byte line that holds the ticket.
constexpr int STATIC_PARTIALS = MAX_PARTIALS;                               // 1024 CTAs at most
constexpr size_t STATIC_TICKET_OFFSET = sizeof(double) * STATIC_PARTIALS;   // 8192
constexpr size_t STATIC_SCRATCH_BYTES = STATIC_TICKET_OFFSET + 256;         // 8448 bytes per GPU
static __device__ __align__(256) unsigned char g_energy_scratch[STATIC_SCRATCH_BYTES];

// In HOST code the name g_energy_scratch is only a handle for the runtime's symbol table, not a
// device address: handing it to a kernel or to cudaMemsetAsync would fault (or, on a system whose
// GPU can reach host memory, quietly use the wrong bytes).  The device address differs per GPU and
// is asked for once per device with cudaGetSymbolAddress, with that device current.
constexpr int STATIC_MAX_DEVICES = 64;
static unsigned char *g_scratch_addr[STATIC_MAX_DEVICES];   // guarded by g_scratch_mutex
static std::mutex g_scratch_mutex;

// The caller has made `device` current.  Returns the scratch address on that device, or nullptr.
static unsigned char *scratch_on_current_device(int device, cudaError_t *err) {
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[device]) {
        void *p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_energy_scratch);
        if (*err != cudaSuccess) return nullptr;
        g_scratch_addr[device] = static_cast<unsigned char *>(p);
    }
    return g_scratch_addr[device];
}

// ---- the kernel --------------------------------------------------------------------------------
// `part` and `ticket` point into g_energy_scratch (device code could name the array itself; taking
// the address as arguments keeps the kernel a plain variant of k_energy).  The ticket must be 0 at
// launch; the last CTA leaves it at 0 again (atomicInc wraps at gridDim.x - 1).
__global__ void __launch_bounds__(RED_THREADS)
k_energy_static(const double *__restrict__ mu, const double *__restrict__ field, long long n3,
                double *__restrict__ part, unsigned *ticket, double *__restrict__ energy) {
    double s = 0, unused = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (long long)gridDim.x * blockDim.x)
        s += mu[i] * field[i];
    block_sum2(s, unused);
    __shared__ bool s_last;
    const int n_part = gridDim.x;
    if (threadIdx.x == 0) {
        part[blockIdx.x] = s;
        __threadfence();
        s_last = atomicInc(ticket, (unsigned)(n_part - 1)) == (unsigned)(n_part - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double x = 0;
    unused = 0;
    for (int i = threadIdx.x; i < n_part; i += RED_THREADS) x += __ldcg(part + i);
    block_sum2(x, unused);
    if (threadIdx.x == 0) *energy = -0.5 * COULOMB * x;
}

struct CurrentDevice {   // make `dev` current for one call and put the caller's device back afterwards
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit CurrentDevice(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) err = cudaSetDevice(dev); else prev = -1;
    }
    ~CurrentDevice() { if (prev >= 0) cudaSetDevice(prev); }
};

static int fail(int code, const char *fmt, long long a = 0, long long b = 0) {
    char msg[256];
    snprintf(msg, sizeof(msg), fmt, a, b);
    set_thread_error(msg);
    return code;
}

}  // namespace tkhp

using namespace tkhp;

extern "C" int tkhp_polar_energy_static(int32_t device, int64_t n_atoms, const double *d_mu, const double *d_field,
                                        double *d_energy, void *stream) {
    if (!d_mu || !d_field || !d_energy) return fail(TKHP_EINVAL, "tkhp_polar_energy_static: NULL argument");
    if (n_atoms < 1) return fail(TKHP_EINVAL, "tkhp_polar_energy_static: n_atoms = %lld, must be >= 1", (long long)n_atoms);
    if (n_atoms > (int64_t)TKHP_STATIC_MAX_ATOMS)
        return fail(TKHP_ECAPACITY,
                    "tkhp_polar_energy_static: n_atoms = %lld exceeds TKHP_STATIC_MAX_ATOMS = %lld (the fixed scratch "
                    "is sized for that; use tkhp_polar_energy on a context for larger systems)",
                    (long long)n_atoms, (long long)TKHP_STATIC_MAX_ATOMS);
    if (device < 0 || device >= STATIC_MAX_DEVICES)
        return fail(TKHP_EINVAL, "tkhp_polar_energy_static: device ordinal %lld outside [0, %lld)", device, STATIC_MAX_DEVICES);
    CurrentDevice cur(device);
    if (cur.err != cudaSuccess) return fail(TKHP_ECUDA, "tkhp_polar_energy_static: cudaSetDevice(%lld) failed", device);
    cudaError_t e = cudaSuccess;
    unsigned char *scratch = scratch_on_current_device(device, &e);   // first call on this device: the set-up
    if (!scratch) {
        char msg[256];
        snprintf(msg, sizeof(msg), "tkhp_polar_energy_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        set_thread_error(msg);
        return TKHP_ECUDA;
    }
    double *part = reinterpret_cast<double *>(scratch);
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + STATIC_TICKET_OFFSET);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const long long n3 = 3LL * n_atoms;
    int g = div_up(n3, RED_THREADS);
    if (g > STATIC_PARTIALS) g = STATIC_PARTIALS;
    // The array is shared by every call and keeps what the last one left.  The partials need no clearing
    // (CTA b writes part[b] before anybody reads it); the ticket must start at 0, and a call that was cut
    // short (a faulting kernel, a reset stream) could have left it elsewhere, so it is cleared every time.
    e = cudaMemsetAsync(ticket, 0, sizeof(unsigned), s);
    if (e == cudaSuccess) {
        k_energy_static<<<g, RED_THREADS, 0, s>>>(d_mu, d_field, n3, part, ticket, d_energy);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof(msg), "tkhp_polar_energy_static: launch failed: %s", cudaGetErrorString(e));
        set_thread_error(msg);
        return TKHP_ECUDA;
    }
    return TKHP_OK;
}
