// Device copy of the term tables of one Hamiltonian (created on first device use) plus library-wide plumbing:
// error text, launch counter, SM count.
#include <atomic>
#include <cstring>
#include <string>
#include <vector>

#include "common.h"

namespace syk {

static thread_local std::string g_cuda_error;
static thread_local int64_t g_launches = 0;

void set_cuda_error(cudaError_t e, const char* what) {
    g_cuda_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " in " + what;
    cudaGetLastError();   // clear the non-sticky error state
}

void count_launch(int n) { g_launches += n; }

// ---- syk_profile_*: event pairs around apply_H launches ----------------------------------------------------
struct ProfileState {
    bool on = false;
    std::vector<cudaEvent_t> ev;   // pairs (begin, end)
    size_t used = 0;               // events recorded
    int64_t untimed = 0;
    bool open = false;
};
static thread_local ProfileState g_prof;
constexpr size_t kMaxProfileEvents = 2 * 65536;

bool profile_enabled() { return g_prof.on; }

uint64_t next_handle_uid() {
    static std::atomic<uint64_t> counter{0};
    return ++counter;
}

void profile_begin(cudaStream_t st) {
    ProfileState& p = g_prof;
    p.open = false;
    if (!p.on) return;
    if (p.used + 2 > kMaxProfileEvents) {
        ++p.untimed;
        return;
    }
    while (p.ev.size() < p.used + 2) {
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) {
            cudaGetLastError();
            ++p.untimed;
            return;
        }
        p.ev.push_back(e);
    }
    if (cudaEventRecord(p.ev[p.used], st) == cudaSuccess) p.open = true;
}

void profile_end(cudaStream_t st) {
    ProfileState& p = g_prof;
    if (!p.open) return;
    p.open = false;
    if (cudaEventRecord(p.ev[p.used + 1], st) == cudaSuccess) p.used += 2;
}

int num_sms() {
    static thread_local int cached_dev = -1, cached = 0;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (dev != cached_dev) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
        cached_dev = dev;
        cached = n;
    }
    return cached;
}

// Tile-load list for tiles of 2^tile_log2 amplitudes: the distinct values of x >> tile_log2 in ascending group
// order.  Load 0 always has hi == 0 (the tile itself; the fused <v|Hv> partial sums need in[b]) even if no
// group lives there.
static void build_load_list(const syk_ham* h, int tile_log2, std::vector<uint32_t>& hi, std::vector<uint32_t>& g0) {
    hi.clear();
    g0.clear();
    hi.push_back(0);
    g0.push_back(0);
    for (size_t g = 0; g < h->x.size(); ++g) {
        uint32_t v = (uint32_t)(h->x[g] >> tile_log2);
        if (v != hi.back()) {
            hi.push_back(v);
            g0.push_back((uint32_t)g);
        }
    }
    g0.push_back((uint32_t)h->x.size());
}

int ensure_device_tables(const syk_ham* h) {
    int dev = 0;
    SYK_CUDA(cudaGetDevice(&dev));
    DeviceTables& d = h->dev;
    if (d.blob && d.device == dev) return SYK_OK;
    if (d.blob) free_device_tables(h);

    const size_t ng = h->x.size(), nt = h->z.size();
    std::vector<uint32_t> hi[2], g0[2];
    for (int k = 0; k < 2; ++k) build_load_list(h, kTileLog2[k], hi[k], g0[k]);

    auto align = [](size_t v) { return (v + 255) & ~(size_t)255; };
    size_t off_gx = 0;
    size_t off_goff = align(off_gx + ng * 4);
    size_t off_tz = align(off_goff + (ng + 1) * 4);
    size_t off_c128 = align(off_tz + nt * 4);
    size_t off_c64 = align(off_c128 + nt * 16);
    size_t off_hi[2], off_g0[2];
    size_t cur = align(off_c64 + nt * 8);
    for (int k = 0; k < 2; ++k) {
        off_hi[k] = cur;
        cur = align(cur + hi[k].size() * 4);
        off_g0[k] = cur;
        cur = align(cur + g0[k].size() * 4);
    }
    const size_t off_sync = cur;
    const size_t total = cur + align(kSyncRing * 4) + 256;

    std::vector<unsigned char> host(total, 0);
    uint32_t* p_gx = (uint32_t*)(host.data() + off_gx);
    uint32_t* p_goff = (uint32_t*)(host.data() + off_goff);
    uint32_t* p_tz = (uint32_t*)(host.data() + off_tz);
    double2* p_c128 = (double2*)(host.data() + off_c128);
    float2* p_c64 = (float2*)(host.data() + off_c64);
    for (size_t g = 0; g < ng; ++g) p_gx[g] = (uint32_t)h->x[g];
    for (size_t g = 0; g <= ng; ++g) p_goff[g] = h->group_off[g];
    for (size_t t = 0; t < nt; ++t) {
        p_tz[t] = (uint32_t)h->z[t];
        p_c128[t] = make_double2(h->c[t].real(), h->c[t].imag());
        p_c64[t] = make_float2((float)h->c[t].real(), (float)h->c[t].imag());
    }
    for (int k = 0; k < 2; ++k) {
        std::memcpy(host.data() + off_hi[k], hi[k].data(), hi[k].size() * 4);
        std::memcpy(host.data() + off_g0[k], g0[k].data(), g0[k].size() * 4);
    }

    void* blob = nullptr;
    SYK_CUDA(cudaMalloc(&blob, total));
    cudaError_t e = cudaMemcpy(blob, host.data(), total, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(blob);
        set_cuda_error(e, "cudaMemcpy(term tables)");
        return SYK_ECUDA;
    }
    unsigned char* b = (unsigned char*)blob;
    d.blob = blob;
    d.device = dev;
    d.gx = (uint32_t*)(b + off_gx);
    d.goff = (uint32_t*)(b + off_goff);
    d.tz = (uint32_t*)(b + off_tz);
    d.tc128 = (double2*)(b + off_c128);
    d.tc64 = (float2*)(b + off_c64);
    d.sync = (uint32_t*)(b + off_sync);
    for (int k = 0; k < 2; ++k) {
        d.load_hi[k] = (uint32_t*)(b + off_hi[k]);
        d.load_g0[k] = (uint32_t*)(b + off_g0[k]);
        d.n_loads[k] = (int)hi[k].size();
    }
    return SYK_OK;
}

void free_device_tables(const syk_ham* h) {
    DeviceTables& d = h->dev;
    if (d.blob) cudaFree(d.blob);
    d = DeviceTables();
}

void invalidate_kernel_tables(const syk_ham* h) {
    free_device_tables(h);
    free_regtile_tables(h);
    free_scatter_tables(h);
    free_dense_tables(h);
    h->dense_representable = -1;
    ++h->table_epoch;
}

}  // namespace syk

extern "C" {

const char* syk_strerror(int code) {
    switch (code) {
        case SYK_OK: return "ok";
        case SYK_EINVAL: return "invalid argument";
        case SYK_ENOMEM: return "work space too small or out of host memory";
        case SYK_ECUDA: return "CUDA error or no CUDA device (see syk_last_cuda_error)";
        case SYK_ENOCONV: return "Krylov sub-step limit reached";
        case SYK_ELIMIT: return "size exceeds the fixed device scratch of a *_static entry point (see syk_dot_static_max_N)";
        default: return "unknown error code";
    }
}

const char* syk_last_cuda_error(void) { return syk::g_cuda_error.c_str(); }

int syk_version(void) { return 100; }

int syk_profile_enable(int on) {
    syk::g_prof.on = on != 0;
    return SYK_OK;
}

int syk_profile_read(double* apply_h_ms, int64_t* apply_h_launches, int reset) {
    syk::ProfileState& p = syk::g_prof;
    double total = 0.0;
    for (size_t i = 0; i + 1 < p.used; i += 2) {
        SYK_CUDA(cudaEventSynchronize(p.ev[i + 1]));
        float ms = 0.f;
        SYK_CUDA(cudaEventElapsedTime(&ms, p.ev[i], p.ev[i + 1]));
        total += ms;
    }
    if (apply_h_ms) *apply_h_ms = total;
    if (apply_h_launches) *apply_h_launches = (int64_t)(p.used / 2);
    if (reset) {
        p.used = 0;
        p.untimed = 0;
    }
    return SYK_OK;
}

int64_t syk_launch_count(int reset) {
    int64_t v = syk::g_launches;
    if (reset) syk::g_launches = 0;
    return v;
}

}  // extern "C"
