// emu_runtime.cpp -- TEST INFRASTRUCTURE: the runtime half of the host emulation (see cuda_runtime.h).
// Memory, deferred streams and events, CUDA arrays, and the fiber scheduler that runs a kernel's CTAs.
#include "cuda_runtime.h"

#include <omp.h>
#include <sys/mman.h>
#include <ucontext.h>

#include <chrono>
#include <cstdio>
#include <deque>
#include <map>
#include <memory>
#include <mutex>
#include <set>
#include <vector>

// =====================================================================================================
// streams and events: queues executed later
// =====================================================================================================
struct emu_event {
    emu_stream* stream = nullptr;          // where the last record was enqueued
    unsigned long long issued = 0;         // records enqueued so far
    unsigned long long done = 0;           // ticket of the last record executed
    double t_ms = 0.0;                     // host clock when the last record executed
};

namespace {

struct Op {
    enum Kind { RUN, RECORD, WAIT } kind;
    std::function<void()> fn;
    emu_event* ev = nullptr;
    unsigned long long ticket = 0;
};

}  // namespace

struct emu_stream {
    std::deque<Op> q;
    bool eager = false;                    // non-blocking (library-private) stream under VR_EMU_SCHED=eager
    bool running = false;                  // re-entrancy guard (a cycle of waits)
};

namespace {

enum Sched { SCHED_SYNC, SCHED_LAZY, SCHED_EAGER };

struct Runtime {
    std::recursive_mutex mu;
    emu_stream legacy;                     // the NULL stream
    std::set<emu_stream*> streams;
    std::map<char*, size_t> pinned;        // cudaHostAlloc ranges
    cudaError_t last = cudaSuccess;
    int max_dyn_smem = 227 * 1024;
    size_t dev_bytes = 0;
    Sched sched = SCHED_LAZY;
    Runtime()
    {
        const char* s = getenv("VR_EMU_SCHED");
        if (s && !strcmp(s, "sync")) sched = SCHED_SYNC;
        if (s && !strcmp(s, "eager")) sched = SCHED_EAGER;
    }
};

Runtime& rt()
{
    static Runtime* r = new Runtime();     // never destroyed: handles may outlive static destruction order
    return *r;
}

double now_ms()
{
    using namespace std::chrono;
    return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

emu_stream* resolve(cudaStream_t s) { return s ? s : &rt().legacy; }

bool run_until(emu_stream* s, emu_event* want, unsigned long long ticket, bool force);

// Executes the ops of `s` in order.  want != null: stops once that record has executed.  force: a WAIT whose record has
// not executed drains the recording stream as far as needed; !force: stops in front of such a WAIT.
// Returns false if it stopped in front of an unsatisfied WAIT.
bool run_until(emu_stream* s, emu_event* want, unsigned long long ticket, bool force)
{
    if (s->running) {
        if (!force) return false;
        fprintf(stderr, "hostemu: a cycle of event waits (deadlock on a real device)\n");
        abort();
    }
    s->running = true;
    bool ok = true;
    while (!s->q.empty()) {
        if (want && want->done >= ticket) break;
        Op& op = s->q.front();
        if (op.kind == Op::WAIT && op.ev->done < op.ticket) {
            if (!force) { ok = false; break; }
            run_until(op.ev->stream, op.ev, op.ticket, true);      // a cycle aborts there
        }
        Op cur = std::move(s->q.front());
        s->q.pop_front();
        if (cur.kind == Op::RUN) cur.fn();
        else if (cur.kind == Op::RECORD) { cur.ev->done = cur.ticket; cur.ev->t_ms = now_ms(); }
    }
    s->running = false;
    return ok;
}

void drain(emu_stream* s) { run_until(s, nullptr, 0, true); }

void drain_all()
{
    drain(&rt().legacy);
    for (emu_stream* s : rt().streams) drain(s);
}

// after every enqueue: what the scheduling policy runs right away
void after_enqueue(emu_stream* s)
{
    Runtime& R = rt();
    if (R.sched == SCHED_SYNC) { drain(s); return; }
    if (R.sched == SCHED_EAGER) {
        // private non-blocking streams run as early as their waits allow; the others as late as possible
        bool progress = true;
        while (progress) {
            progress = false;
            for (emu_stream* e : R.streams)
                if (e->eager && !e->q.empty()) {
                    const size_t before = e->q.size();
                    run_until(e, nullptr, 0, false);
                    progress = progress || e->q.size() != before;
                }
        }
    }
}

void enqueue(cudaStream_t s, std::function<void()> fn)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    emu_stream* st = resolve(s);
    Op op; op.kind = Op::RUN; op.fn = std::move(fn);
    st->q.push_back(std::move(op));
    after_enqueue(st);
}

bool is_pinned(const void* p, size_t bytes)
{
    Runtime& R = rt();
    auto it = R.pinned.upper_bound((char*)p);
    if (it == R.pinned.begin()) return false;
    --it;
    return (char*)p + bytes <= it->first + it->second;
}

}  // namespace

const char* cudaGetErrorString(cudaError_t e)
{
    switch (e) {
    case cudaSuccess: return "no error";
    case cudaErrorInvalidValue: return "invalid argument";
    case cudaErrorMemoryAllocation: return "out of memory";
    case cudaErrorInvalidDevice: return "invalid device ordinal";
    case cudaErrorNotReady: return "device not ready";
    default: return "unspecified launch failure";
    }
}

cudaError_t cudaGetLastError() { cudaError_t e = rt().last; rt().last = cudaSuccess; return e; }
// VR_EMU_DEVICES (default 1): how many "devices" there are; they are all this process' host memory
static int emu_device_count()
{
    const char* e = getenv("VR_EMU_DEVICES");
    const int n = e ? atoi(e) : 1;
    return n >= 1 ? n : 1;
}
cudaError_t cudaGetDeviceCount(int* n) { *n = emu_device_count(); return cudaSuccess; }
cudaError_t cudaSetDevice(int d) { return d >= 0 && d < emu_device_count() ? cudaSuccess : cudaErrorInvalidDevice; }
cudaError_t cudaMemGetInfo(size_t* f, size_t* t) { *t = (size_t)180 << 30; *f = *t - rt().dev_bytes; return cudaSuccess; }

cudaError_t cudaMalloc(void** p, size_t bytes)
{
    *p = nullptr;
    if (bytes == 0) bytes = 1;
    void* q = nullptr;
    if (posix_memalign(&q, 256, (bytes + 255) / 256 * 256) != 0) return rt().last = cudaErrorMemoryAllocation;
    memset(q, 0xA5, bytes);                // device memory is never zero-initialised
    *p = q;
    return cudaSuccess;
}

cudaError_t cudaFree(void* p)
{
    if (!p) return cudaSuccess;
    { std::lock_guard<std::recursive_mutex> g(rt().mu); drain_all(); }     // cudaFree synchronises the device
    free(p);
    return cudaSuccess;
}

cudaError_t cudaHostAlloc(void** p, size_t bytes, unsigned int)
{
    *p = nullptr;
    void* q = nullptr;
    if (posix_memalign(&q, 4096, (bytes + 4095) / 4096 * 4096) != 0) return rt().last = cudaErrorMemoryAllocation;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    rt().pinned[(char*)q] = bytes;
    *p = q;
    return cudaSuccess;
}

cudaError_t cudaFreeHost(void* p)
{
    if (!p) return cudaSuccess;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();
    rt().pinned.erase((char*)p);
    free(p);
    return cudaSuccess;
}

cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t bytes, cudaMemcpyKind kind, cudaStream_t s)
{
    if (bytes == 0) return cudaSuccess;
    if (!dst || !src) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    if (kind == cudaMemcpyHostToDevice && !is_pinned(src, bytes)) {
        // pageable source: the runtime stages it before returning
        std::shared_ptr<std::vector<char>> tmp = std::make_shared<std::vector<char>>((const char*)src, (const char*)src + bytes);
        enqueue(s, [dst, tmp]() { memcpy(dst, tmp->data(), tmp->size()); });
        return cudaSuccess;
    }
    if (kind == cudaMemcpyDeviceToHost && !is_pinned(dst, bytes)) {
        // pageable destination: the call returns once the copy has completed
        drain(resolve(s));
        memcpy(dst, src, bytes);
        return cudaSuccess;
    }
    enqueue(s, [dst, src, bytes]() { memmove(dst, src, bytes); });
    return cudaSuccess;
}

cudaError_t cudaMemcpy(void* dst, const void* src, size_t bytes, cudaMemcpyKind)
{
    if (bytes == 0) return cudaSuccess;
    if (!dst || !src) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();
    memmove(dst, src, bytes);
    return cudaSuccess;
}

cudaError_t cudaMemsetAsync(void* p, int value, size_t bytes, cudaStream_t s)
{
    if (!p && bytes) return rt().last = cudaErrorInvalidValue;
    enqueue(s, [p, value, bytes]() { memset(p, value, bytes); });
    return cudaSuccess;
}

cudaError_t cudaMemset(void* p, int value, size_t bytes)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();
    memset(p, value, bytes);
    return cudaSuccess;
}

cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned int flags)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    emu_stream* st = new emu_stream();
    st->eager = (flags & cudaStreamNonBlocking) != 0;
    rt().streams.insert(st);
    *s = st;
    return cudaSuccess;
}

cudaError_t cudaStreamDestroy(cudaStream_t s)
{
    if (!s) return cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain(s);
    rt().streams.erase(s);
    delete s;
    return cudaSuccess;
}

cudaError_t cudaStreamSynchronize(cudaStream_t s)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain(resolve(s));
    return cudaSuccess;
}

cudaError_t cudaDeviceSynchronize()
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();
    return cudaSuccess;
}

cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned int) { *e = new emu_event(); return cudaSuccess; }

cudaError_t cudaEventDestroy(cudaEvent_t e)
{
    if (!e) return cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();                            // queued records / waits still name it
    delete e;
    return cudaSuccess;
}

cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s)
{
    if (!e) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    emu_stream* st = resolve(s);
    Op op; op.kind = Op::RECORD; op.ev = e; op.ticket = ++e->issued;
    e->stream = st;
    st->q.push_back(std::move(op));
    after_enqueue(st);
    return cudaSuccess;
}

cudaError_t cudaStreamWaitEvent(cudaStream_t s, cudaEvent_t e, unsigned int)
{
    if (!e) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    if (e->issued == 0) return cudaSuccess;            // never recorded: the wait is a no-op
    emu_stream* st = resolve(s);
    Op op; op.kind = Op::WAIT; op.ev = e; op.ticket = e->issued;   // the most recent record at the time of the call
    st->q.push_back(std::move(op));
    after_enqueue(st);
    return cudaSuccess;
}

cudaError_t cudaEventSynchronize(cudaEvent_t e)
{
    if (!e) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    if (e->issued && e->done < e->issued) run_until(e->stream, e, e->issued, true);
    return cudaSuccess;
}

cudaError_t cudaEventQuery(cudaEvent_t e)
{
    if (!e) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    return e->done >= e->issued ? cudaSuccess : cudaErrorNotReady;
}

cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b)
{
    if (!a || !b || !ms) return rt().last = cudaErrorInvalidValue;
    if (a->done < a->issued || b->done < b->issued) return cudaErrorNotReady;
    *ms = (float)(b->t_ms - a->t_ms);
    return cudaSuccess;
}

// =====================================================================================================
// CUDA arrays, texture objects
// =====================================================================================================
cudaError_t cudaMalloc3DArray(cudaArray_t* arr, const cudaChannelFormatDesc*, cudaExtent ext, unsigned int flags)
{
    *arr = nullptr;
    if (!(flags & cudaArrayLayered) || ext.width == 0 || ext.height == 0 || ext.depth == 0) return rt().last = cudaErrorInvalidValue;
    if (ext.width > 32768 || ext.height > 32768 || ext.depth > 2048) return rt().last = cudaErrorInvalidValue;   // maxTexture2DLayered
    cudaArray* a = new cudaArray();
    a->w = (int)ext.width; a->h = (int)ext.height; a->layers = (int)ext.depth;
    const size_t n = ext.width * ext.height * ext.depth;
    a->data = (float*)malloc(n * sizeof(float));
    if (!a->data) { delete a; return rt().last = cudaErrorMemoryAllocation; }
    memset(a->data, 0xA5, n * sizeof(float));
    *arr = a;
    return cudaSuccess;
}

cudaError_t cudaFreeArray(cudaArray_t a)
{
    if (!a) return cudaSuccess;
    { std::lock_guard<std::recursive_mutex> g(rt().mu); drain_all(); }
    free(a->data);
    delete a;
    return cudaSuccess;
}

cudaError_t cudaCreateTextureObject(cudaTextureObject_t* tex, const cudaResourceDesc* rd, const cudaTextureDesc* td, const void*)
{
    if (!rd || !td || rd->resType != cudaResourceTypeArray || !rd->res.array.array) return rt().last = cudaErrorInvalidValue;
    if (td->filterMode != cudaFilterModePoint || td->normalizedCoords || td->addressMode[0] != cudaAddressModeClamp ||
        td->addressMode[1] != cudaAddressModeClamp)
        return rt().last = cudaErrorInvalidValue;          // the only kind the emulated gather models
    *tex = (cudaTextureObject_t)(uintptr_t)rd->res.array.array;
    return cudaSuccess;
}

cudaError_t cudaDestroyTextureObject(cudaTextureObject_t) { return cudaSuccess; }

cudaError_t cudaMemcpy3DAsync(const cudaMemcpy3DParms* pp, cudaStream_t s)
{
    if (!pp) return rt().last = cudaErrorInvalidValue;
    const cudaMemcpy3DParms p = *pp;
    if (p.srcArray) return rt().last = cudaErrorInvalidValue;   // not used by the library
    if (!p.srcPtr.ptr) return rt().last = cudaErrorInvalidValue;
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    // when an array takes part, extent and positions are in elements; else in bytes along x
    const size_t esz = p.dstArray ? sizeof(float) : 1;
    const size_t row_bytes = p.extent.width * esz;
    const size_t src_bytes = ((p.extent.depth - 1) * p.srcPtr.ysize + (p.extent.height - 1)) * p.srcPtr.pitch + row_bytes;
    const char* src0 = (const char*)p.srcPtr.ptr + (p.srcPos.z * p.srcPtr.ysize + p.srcPos.y) * p.srcPtr.pitch + p.srcPos.x * esz;
    std::shared_ptr<std::vector<char>> staged;
    if (p.kind == cudaMemcpyHostToDevice && !is_pinned(src0, src_bytes)) {
        staged = std::make_shared<std::vector<char>>(src0, src0 + src_bytes);
        src0 = nullptr;
    }
    if (p.dstArray) {
        cudaArray_t a = p.dstArray;
        if (p.dstPos.x + p.extent.width > (size_t)a->w || p.dstPos.y + p.extent.height > (size_t)a->h ||
            p.dstPos.z + p.extent.depth > (size_t)a->layers)
            return rt().last = cudaErrorInvalidValue;
    } else if (!p.dstPtr.ptr) {
        return rt().last = cudaErrorInvalidValue;
    }
    enqueue(s, [p, src0, staged, row_bytes, esz]() {
        const char* src = staged ? staged->data() : src0;
        for (size_t z = 0; z < p.extent.depth; ++z)
            for (size_t y = 0; y < p.extent.height; ++y) {
                const char* sr = src + (z * p.srcPtr.ysize + y) * p.srcPtr.pitch;
                char* dr;
                if (p.dstArray) {
                    cudaArray_t a = p.dstArray;
                    dr = (char*)(a->data + ((p.dstPos.z + z) * (size_t)a->h + (p.dstPos.y + y)) * (size_t)a->w + p.dstPos.x);
                } else {
                    dr = (char*)p.dstPtr.ptr + ((p.dstPos.z + z) * p.dstPtr.ysize + (p.dstPos.y + y)) * p.dstPtr.pitch + p.dstPos.x * esz;
                }
                memcpy(dr, sr, row_bytes);
            }
    });
    return cudaSuccess;
}

namespace emu {

float4 tld4_a2d(cudaTextureObject_t tex, int layer, float x, float y)
{
    const cudaArray* a = (const cudaArray*)(uintptr_t)tex;
    // unnormalised coordinates: the bilinear footprint of (x, y) starts at texel floor(x - 0.5), floor(y - 0.5)
    const int i0 = (int)floorf(x - 0.5f), j0 = (int)floorf(y - 0.5f);
    auto cl = [](int v, int n) { return v < 0 ? 0 : (v >= n ? n - 1 : v); };
    const int l = cl(layer, a->layers);
    const int i[2] = {cl(i0, a->w), cl(i0 + 1, a->w)}, j[2] = {cl(j0, a->h), cl(j0 + 1, a->h)};
    const float* L = a->data + (size_t)l * a->h * a->w;
    // counter-clockwise from the lower-left of the footprint: (i, j+1), (i+1, j+1), (i+1, j), (i, j)
    return make_float4(L[(size_t)j[1] * a->w + i[0]], L[(size_t)j[1] * a->w + i[1]], L[(size_t)j[0] * a->w + i[1]],
                       L[(size_t)j[0] * a->w + i[0]]);
}

// =====================================================================================================
// kernels: one CTA = a set of fibers on one OS thread
// =====================================================================================================
thread_local ThreadInfo* g_thr = nullptr;
thread_local BlockInfo* g_blk = nullptr;

namespace {

constexpr size_t kStackBytes = 256 * 1024;

struct Fiber {
    ucontext_t uc;
    char* stack = nullptr;
    ThreadInfo info;
    bool done = false;
    int warp = 0, lane = 0;
};

struct Warp {
    unsigned int vals[32];
    unsigned int present = 0;
    int alive = 0, arrived = 0;
    unsigned int gen = 0;
};

struct Cta {
    BlockInfo info;
    std::vector<Fiber> fibers;
    std::vector<Warp> warps;
    ucontext_t sched;
    Fiber* cur = nullptr;
    int alive = 0, arrived = 0;
    unsigned int gen = 0;
    std::vector<char> dyn;
    const std::function<void()>* body = nullptr;
    unsigned long long switches = 0;
};

thread_local Cta* t_cta = nullptr;

void yield_fiber()
{
    Cta* c = t_cta;
    ++c->switches;
    swapcontext(&c->cur->uc, &c->sched);
}

void release_if_complete(Cta* c)
{
    if (c->alive > 0 && c->arrived == c->alive) { c->arrived = 0; ++c->gen; }
}

void release_warp_if_complete(Warp& w)
{
    if (w.alive > 0 && w.arrived == w.alive) { w.arrived = 0; ++w.gen; }
}

void warp_barrier(Cta* c, Warp& w)
{
    const unsigned int g = w.gen;
    ++w.arrived;
    release_warp_if_complete(w);
    while (w.gen == g) yield_fiber();
    (void)c;
}

void trampoline()
{
    Cta* c = t_cta;
    (*c->body)();
    Fiber* f = c->cur;
    f->done = true;
    // an exited thread takes no part in later barriers / collectives
    --c->alive;
    release_if_complete(c);
    Warp& w = c->warps[f->warp];
    --w.alive;
    w.present &= ~(1u << f->lane);
    release_warp_if_complete(w);
    swapcontext(&f->uc, &c->sched);
}

void run_cta(Cta* c, unsigned int bx, unsigned int by, unsigned int bz, size_t smem)
{
    c->info.bid = uint3{bx, by, bz};
    const dim3 b = c->info.block;
    const int n = (int)(b.x * b.y * b.z);
    if ((int)c->fibers.size() < n) {
        const size_t old = c->fibers.size();
        c->fibers.resize(n);
        for (size_t q = old; q < (size_t)n; ++q) {
            void* st = mmap(nullptr, kStackBytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS | MAP_NORESERVE, -1, 0);
            if (st == MAP_FAILED) { fprintf(stderr, "hostemu: cannot map a fiber stack\n"); abort(); }
            c->fibers[q].stack = (char*)st;
        }
    }
    c->warps.assign((n + 31) / 32, Warp());
    c->alive = n; c->arrived = 0; c->gen = 0;
    c->dyn.assign(smem + 16, 0);
    // uninitialised shared memory: NaNs
    {
        float* d = (float*)(((uintptr_t)c->dyn.data() + 15) & ~(uintptr_t)15);
        for (size_t q = 0; q < smem / 4; ++q) d[q] = NAN;
    }
    for (int t = 0; t < n; ++t) {
        Fiber& f = c->fibers[t];
        f.done = false;
        f.info.tid = uint3{(unsigned)t % b.x, ((unsigned)t / b.x) % b.y, (unsigned)t / (b.x * b.y)};
        f.warp = t >> 5; f.lane = t & 31;
        Warp& w = c->warps[f.warp];
        ++w.alive; w.present |= 1u << f.lane;
        getcontext(&f.uc);
        f.uc.uc_stack.ss_sp = f.stack;
        f.uc.uc_stack.ss_size = kStackBytes;
        f.uc.uc_link = &c->sched;
        makecontext(&f.uc, (void (*)())trampoline, 0);
    }
    g_blk = &c->info;
    int remaining = n;
    unsigned long long idle_passes = 0;
    while (remaining > 0) {
        int progressed = 0;
        for (int t = 0; t < n; ++t) {
            Fiber& f = c->fibers[t];
            if (f.done) continue;
            c->cur = &f;
            g_thr = &f.info;
            const unsigned int g0 = c->gen;
            swapcontext(&c->sched, &f.uc);
            if (f.done) { --remaining; ++progressed; }
            else if (c->gen != g0) ++progressed;
        }
        // a pass in which nothing finished and no barrier opened may still be progress (warp collectives); a very long
        // run of them is a deadlock: threads waiting at a barrier that others never reach
        idle_passes = progressed ? 0 : idle_passes + 1;
        if (idle_passes > 1000000ull) { fprintf(stderr, "hostemu: CTA deadlock (divergent barrier?)\n"); abort(); }
    }
    g_thr = nullptr;
}

}  // namespace

void* dyn_smem()
{
    return (void*)(((uintptr_t)t_cta->dyn.data() + 15) & ~(uintptr_t)15);
}

void yield() { yield_fiber(); }

void syncthreads()
{
    Cta* c = t_cta;
    const unsigned int g = c->gen;
    ++c->arrived;
    release_if_complete(c);
    while (c->gen == g) yield_fiber();
}

int warp_exchange(unsigned int v, unsigned int all[32], unsigned int* present)
{
    Cta* c = t_cta;
    Fiber* f = c->cur;
    Warp& w = c->warps[f->warp];
    w.vals[f->lane] = v;
    warp_barrier(c, w);
    for (int l = 0; l < 32; ++l) all[l] = w.vals[l];
    *present = w.present;
    warp_barrier(c, w);                     // nobody overwrites a value before everybody has read it
    return f->lane;
}

cudaError_t set_max_dyn_smem(int bytes)
{
    return bytes <= 227 * 1024 ? cudaSuccess : (rt().last = cudaErrorInvalidValue);
}

cudaError_t enqueue_kernel(cudaStream_t s, dim3 grid, dim3 block, size_t smem, std::function<void()> body)
{
    const unsigned long long nthreads = (unsigned long long)block.x * block.y * block.z;
    if (nthreads == 0 || nthreads > 1024 || grid.x == 0 || grid.y == 0 || grid.z == 0 || grid.y > 65535 || grid.z > 65535 ||
        smem > 227 * 1024)
        return rt().last = cudaErrorInvalidValue;          // "invalid configuration argument"
    std::shared_ptr<std::function<void()>> fn = std::make_shared<std::function<void()>>(std::move(body));
    enqueue(s, [grid, block, smem, fn]() {
        const long long nblocks = (long long)grid.x * grid.y * grid.z;
        const int want = getenv("VR_EMU_THREADS") ? atoi(getenv("VR_EMU_THREADS")) : omp_get_max_threads();
#pragma omp parallel num_threads(want > 0 ? want : 1)
        {
            static thread_local Cta* cta = nullptr;        // fibers and stacks are reused from launch to launch
            if (!cta) cta = new Cta();
            cta->info.grid = grid;
            cta->info.block = block;
            cta->body = fn.get();
            t_cta = cta;
#pragma omp for schedule(dynamic, 1)
            for (long long q = 0; q < nblocks; ++q)
                run_cta(cta, (unsigned)(q % grid.x), (unsigned)((q / grid.x) % grid.y), (unsigned)(q / ((long long)grid.x * grid.y)), smem);
            g_blk = nullptr;
        }
    });
    return cudaSuccess;
}

}  // namespace emu

// ---- hooks for the tests (tests/backends.py) -------------------------------------------------------------
extern "C" {

// everything enqueued so far has run when this returns
void vr_emu_sync(void) { cudaDeviceSynchronize(); }

// 0 = sync, 1 = lazy, 2 = eager (see cuda_runtime.h); takes effect for later enqueues
void vr_emu_set_sched(int mode)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    drain_all();
    rt().sched = mode == 0 ? SCHED_SYNC : (mode == 2 ? SCHED_EAGER : SCHED_LAZY);
}

// ops still queued in all streams (a test can see that work really was deferred)
unsigned long long vr_emu_pending(void)
{
    std::lock_guard<std::recursive_mutex> g(rt().mu);
    unsigned long long n = rt().legacy.q.size();
    for (emu_stream* s : rt().streams) n += s->q.size();
    return n;
}

}  // extern "C"
