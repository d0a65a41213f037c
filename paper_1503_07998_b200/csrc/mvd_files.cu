// mvd_files.cu -- disk I/O as the outer stage of the pipeline (Supp. Note 2 s.3, Algorithm 1:
// "not only copies to and from the GPU, but also loading and saving data from and to hard-drive come without
// additional cost").  Algorithm 1 cycles single planes through three streams; here SLABS of planes cycle through three
// pinned buffer sets: while slab k runs through mvd_deconvolve_host_ex (itself the 3-stream H2D / RL / D2H pipeline), a
// reader thread loads slab k + 1 from the view files and a writer thread saves slab k - 1.
#include <fcntl.h>
#include <string.h>
#include <sys/stat.h>
#include <unistd.h>

#include <algorithm>
#include <condition_variable>
#include <mutex>
#include <thread>
#include <vector>

#include "mvd_internal.cuh"

namespace {

bool read_fully(int fd, void* dst, size_t bytes, off_t off) {
    char* p = static_cast<char*>(dst);
    while (bytes) {
        const ssize_t r = pread(fd, p, bytes, off);
        if (r <= 0) return false;
        p += r; off += r; bytes -= (size_t)r;
    }
    return true;
}
bool write_fully(int fd, const void* src, size_t bytes, off_t off) {
    const char* p = static_cast<const char*>(src);
    while (bytes) {
        const ssize_t r = pwrite(fd, p, bytes, off);
        if (r <= 0) return false;
        p += r; off += r; bytes -= (size_t)r;
    }
    return true;
}

// One slot of the three-deep ring: LOADING -> LOADED -> COMPUTED -> (saved) FREE
struct Slot {
    uint16_t* in = nullptr;
    void* out = nullptr;
    int p0 = 0, n = 0;
    enum State { FREE, LOADED, COMPUTED } state = FREE;
};

}  // namespace

int mvd_deconvolve_files(mvd_handle* h, const char* const* view_paths, const char* out_path, int n_planes, int out_type) {
    if (!h || !view_paths || !out_path || n_planes < 0) return MVD_ERR_INVALID;
    if (out_type != MVD_OUT_F32 && out_type != MVD_OUT_U16) return MVD_ERR_INVALID;
    for (int v = 0; v < h->V; ++v)
        if (!view_paths[v]) return MVD_ERR_INVALID;
    if (n_planes == 0) return MVD_OK;
    const size_t npx = (size_t)h->uW * h->uH;
    const size_t out_elem = out_type == MVD_OUT_U16 ? sizeof(uint16_t) : sizeof(float);

    // slab: a whole number of pipeline batches, about 256 MiB of input, at least four slabs when the stack allows it
    const int B = std::max(2, mvd_get_batch_planes(h, n_planes));
    size_t slab = std::max<size_t>(1, ((size_t)256 << 20) / (npx * sizeof(uint16_t) * h->V));
    slab = std::min<size_t>(slab, (size_t)std::max(1, n_planes / 4));
    slab = std::max<size_t>((slab / B) * B, (size_t)B);          // even for the FFT engine's plane pairing (B is)
    slab = std::min<size_t>(slab, (size_t)n_planes);
    const int S = (int)slab;

    std::vector<int> fds(h->V, -1);
    int ofd = -1;
    int rc = MVD_OK;
    for (int v = 0; v < h->V && rc == MVD_OK; ++v) {
        fds[v] = open(view_paths[v], O_RDONLY);
        struct stat st;
        if (fds[v] < 0 || fstat(fds[v], &st) != 0 || (size_t)st.st_size < npx * sizeof(uint16_t) * n_planes) rc = MVD_ERR_IO;
    }
    if (rc == MVD_OK) {
        ofd = open(out_path, O_WRONLY | O_CREAT | O_TRUNC, 0644);
        if (ofd < 0) rc = MVD_ERR_IO;
    }
    Slot slots[3];
    for (int k = 0; k < 3 && rc == MVD_OK; ++k) {
        rc = mvd_check(h, cudaHostAlloc((void**)&slots[k].in, npx * sizeof(uint16_t) * S * h->V, cudaHostAllocDefault));
        if (rc == MVD_OK) rc = mvd_check(h, cudaHostAlloc(&slots[k].out, npx * out_elem * S, cudaHostAllocDefault));
    }

    if (rc == MVD_OK) {
        std::mutex mu;
        std::condition_variable cv;
        bool failed = false;
        const int n_slabs = (n_planes + S - 1) / S;
        // reader: slab k -> slot k % 3 as soon as that slot is free        (Algorithm 1: "Load plane z from hard-drive")
        std::thread reader([&] {
            for (int k = 0; k < n_slabs; ++k) {
                Slot& s = slots[k % 3];
                {
                    std::unique_lock<std::mutex> lk(mu);
                    cv.wait(lk, [&] { return s.state == Slot::FREE || failed; });
                    if (failed) return;
                }
                s.p0 = k * S;
                s.n = std::min(S, n_planes - s.p0);
                bool ok = true;
                for (int v = 0; v < h->V && ok; ++v)     // the slab's planes of view v, packed [V][n][H][W]
                    ok = read_fully(fds[v], s.in + (size_t)v * s.n * npx, npx * sizeof(uint16_t) * s.n,
                                    (off_t)((size_t)s.p0 * npx * sizeof(uint16_t)));
                std::lock_guard<std::mutex> lk(mu);
                if (!ok) failed = true;
                else s.state = Slot::LOADED;
                cv.notify_all();
                if (!ok) return;
            }
        });
        // writer: slab k from slot k % 3 once it is computed                (Algorithm 1: "Save deconvolved plane")
        std::thread writer([&] {
            for (int k = 0; k < n_slabs; ++k) {
                Slot& s = slots[k % 3];
                {
                    std::unique_lock<std::mutex> lk(mu);
                    cv.wait(lk, [&] { return s.state == Slot::COMPUTED || failed; });
                    if (failed) return;
                }
                const bool ok = write_fully(ofd, s.out, npx * out_elem * s.n, (off_t)((size_t)s.p0 * npx * out_elem));
                std::lock_guard<std::mutex> lk(mu);
                if (!ok) failed = true;
                else s.state = Slot::FREE;
                cv.notify_all();
                if (!ok) return;
            }
        });
        // this thread: the GPU pipeline on slab k                            (Algorithm 1: H2D, RL steps, D2H)
        for (int k = 0; k < n_slabs; ++k) {
            Slot& s = slots[k % 3];
            {
                std::unique_lock<std::mutex> lk(mu);
                cv.wait(lk, [&] { return s.state == Slot::LOADED || failed; });
                if (failed) break;
            }
            const mvd_io io = {s.in, 0, 0, 0, nullptr, s.out, out_type, 0};
            const int r = mvd_deconvolve_host_ex(h, &io, s.n);
            std::lock_guard<std::mutex> lk(mu);
            if (r != MVD_OK) { rc = r; failed = true; }
            else s.state = Slot::COMPUTED;
            cv.notify_all();
            if (r != MVD_OK) break;
        }
        reader.join();
        writer.join();
        if (failed && rc == MVD_OK) rc = MVD_ERR_IO;
    }
    for (int k = 0; k < 3; ++k) {
        if (slots[k].in) cudaFreeHost(slots[k].in);
        if (slots[k].out) cudaFreeHost(slots[k].out);
    }
    for (int fd : fds)
        if (fd >= 0) close(fd);
    if (ofd >= 0 && close(ofd) != 0 && rc == MVD_OK) rc = MVD_ERR_IO;
    return rc;
}
