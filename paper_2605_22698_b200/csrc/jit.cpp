// NVRTC compilation of the generated kernels to an sm_100a cubin and loading through the CUDA
// runtime's library API (no driver-API link dependency, so the .so also loads on a box without
// a GPU driver, where it is only ever used for the build check).
#include <nvrtc.h>
#include <sys/stat.h>
#include <unistd.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <string>

#include "e3_internal.h"

namespace e3 {

static int parse_after(const std::string &log, const std::string &fn, const char *key_before, const char *key)
{
    // finds "... <number> <key>" inside the ptxas block of function fn
    size_t pos = log.find("Function properties for " + fn);
    if (pos == std::string::npos) pos = 0;
    (void)key_before;
    size_t k = log.find(key, pos);
    if (k == std::string::npos) return -1;
    size_t b = k;
    while (b > 0 && (log[b - 1] == ' ')) --b;
    size_t a = b;
    while (a > 0 && log[a - 1] >= '0' && log[a - 1] <= '9') --a;
    if (a == b) return -1;
    return atoi(log.substr(a, b - a).c_str());
}

// FNV-1a, 64 bit: a second, independent hash beside std::hash (the cache key carries both)
static unsigned long long fnv1a64(const std::string &s)
{
    unsigned long long h = 1469598103934665603ULL;
    for (unsigned char c : s) { h ^= c; h *= 1099511628211ULL; }
    return h;
}

static const char *kNvrtcOpts[] = { "--gpu-architecture=sm_100a", "-lineinfo", "--std=c++17", "--ptxas-options=-v", "-default-device" };

// Per-user cache directory (mode 0700, owned by the caller, not a symlink): $E3_JIT_DIR, else $XDG_CACHE_HOME/e3b200_jit,
// else /tmp/e3b200_jit_<uid>.  Returns "" when no safe directory can be had (the cache is then simply not used).
static std::string jit_dir()
{
    std::string dir;
    if (const char *d = getenv("E3_JIT_DIR")) dir = d;
    else if (const char *x = getenv("XDG_CACHE_HOME")) dir = std::string(x) + "/e3b200_jit";
    else dir = "/tmp/e3b200_jit_" + std::to_string((long)getuid());
    mkdir(dir.c_str(), 0700);
    struct stat st;
    if (lstat(dir.c_str(), &st) != 0 || !S_ISDIR(st.st_mode) || st.st_uid != getuid() || (st.st_mode & 022)) return "";
    return dir;
}

static bool read_file(const std::string &path, std::string &out)
{
    FILE *f = fopen(path.c_str(), "rb");
    if (!f) return false;
    out.clear();
    char buf[65536];
    size_t n;
    while ((n = fread(buf, 1, sizeof(buf), f)) > 0) out.append(buf, n);
    fclose(f);
    return true;
}

int jit_compile(JitKernel &k, const std::string &file_hint)
{
    // keep the generated source on disk so that -lineinfo maps SASS back to it (ncu source page)
    const std::string dir = jit_dir();
    std::string opt_key;
    for (const char *o : kNvrtcOpts) { opt_key += o; opt_key += '\n'; }
    const std::string keyed = opt_key + k.source;
    char hb[64];
    snprintf(hb, sizeof(hb), "%016zx%016llx", std::hash<std::string>{}(keyed), fnv1a64(keyed));
    std::string path = file_hint.empty() ? (dir.empty() ? std::string("e3_jit_") + k.name + ".cu" : dir + "/" + k.name + "_" + hb + ".cu") : file_hint;

    // compiled-code cache (speed only).  Key: two independent 64-bit hashes of (compile options + generated source), the
    // source length and the NVRTC version.  A hit is accepted only if the source stored beside the cubin is byte-identical
    // to the generated one and the cubin matches the length and checksum recorded in the .info file.  E3_JIT_CACHE=0 disables it.
    int vmaj = 0, vmin = 0;
    nvrtcVersion(&vmaj, &vmin);
    char vb[64];
    snprintf(vb, sizeof(vb), "_%zu_nvrtc%d_%d", k.source.size(), vmaj, vmin);
    const char *cache_env = getenv("E3_JIT_CACHE");
    const bool use_cache = !(cache_env && cache_env[0] == '0') && file_hint.empty() && !dir.empty();
    const std::string cpath = dir + "/" + k.name + "_" + hb + vb + ".cubin", ipath = cpath + ".info";
    if (use_cache) {
        std::string stored_src, info, cub;
        long long want = -1;
        unsigned long long sum = 0;
        int regs = 0, spill = 0, smem = 0;
        if (read_file(path, stored_src) && stored_src == k.source && read_file(ipath, info) && read_file(cpath, cub) &&
            sscanf(info.c_str(), "%lld %d %d %d %llx", &want, &regs, &spill, &smem, &sum) == 5 && want > 0 &&
            (size_t)want == cub.size() && sum == fnv1a64(cub)) {
            k.cubin.assign(cub.begin(), cub.end());
            k.regs = regs; k.spill = spill; k.smem = smem;
            return E3_OK;
        }
    }
    if (file_hint.empty() ? !dir.empty() : true)
        if (FILE *f = fopen(path.c_str(), "w")) { fwrite(k.source.data(), 1, k.source.size(), f); fclose(f); }

    nvrtcProgram prog;
    if (nvrtcCreateProgram(&prog, k.source.c_str(), path.c_str(), 0, nullptr, nullptr) != NVRTC_SUCCESS) {
        set_error("nvrtcCreateProgram failed");
        return E3_ERR_JIT;
    }
    const char *cuda_home = getenv("CUDA_HOME");
    std::string inc = std::string("-I") + (cuda_home ? cuda_home : "/usr/local/cuda") + "/include";
    const char *opts[] = { kNvrtcOpts[0], kNvrtcOpts[1], kNvrtcOpts[2], kNvrtcOpts[3], kNvrtcOpts[4], inc.c_str() };
    nvrtcResult r = nvrtcCompileProgram(prog, 6, opts);
    size_t ls = 0;
    nvrtcGetProgramLogSize(prog, &ls);
    std::string log(ls, '\0');
    if (ls) nvrtcGetProgramLog(prog, &log[0]);
    if (r != NVRTC_SUCCESS) {
        set_error("NVRTC failed for %s (%s):\n%.12000s", k.name.c_str(), nvrtcGetErrorString(r), log.c_str());
        nvrtcDestroyProgram(&prog);
        return E3_ERR_JIT;
    }
    size_t cs = 0;
    nvrtcGetCUBINSize(prog, &cs);
    k.cubin.resize(cs);
    nvrtcGetCUBIN(prog, k.cubin.data());
    nvrtcDestroyProgram(&prog);
    k.regs = parse_after(log, k.name, "Used", "registers");
    k.spill = parse_after(log, k.name, "stack frame,", "bytes spill stores");
    int sm = parse_after(log, k.name, ",", "bytes smem");
    k.smem = sm < 0 ? 0 : sm;
    if (use_cache) {      // write to a temporary name and rename: concurrent processes (one per GPU) may build the same plan
        char tb[64];
        snprintf(tb, sizeof(tb), ".tmp%ld", (long)getpid());
        const std::string tc = cpath + tb, ti = ipath + tb;
        FILE *fc = fopen(tc.c_str(), "wb"), *fi = fopen(ti.c_str(), "w");
        bool ok = fc && fi && fwrite(k.cubin.data(), 1, k.cubin.size(), fc) == k.cubin.size() &&
                  fprintf(fi, "%lld %d %d %d %llx\n", (long long)k.cubin.size(), k.regs, k.spill, k.smem,
                          fnv1a64(std::string(k.cubin.begin(), k.cubin.end()))) > 0;
        if (fc) fclose(fc);
        if (fi) fclose(fi);
        if (ok) ok = rename(tc.c_str(), cpath.c_str()) == 0 && rename(ti.c_str(), ipath.c_str()) == 0;
        if (!ok) { remove(tc.c_str()); remove(ti.c_str()); }
    }
    if (!file_hint.empty()) {
        std::string cp = file_hint + ".cubin";
        if (FILE *f = fopen(cp.c_str(), "wb")) { fwrite(k.cubin.data(), 1, k.cubin.size(), f); fclose(f); }
    }
    return E3_OK;
}

int jit_load(JitKernel &k)
{
    if (k.fn) return E3_OK;
    E3_CUDA_TRY(cudaLibraryLoadData(&k.lib, k.cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0));
    E3_CUDA_TRY(cudaLibraryGetKernel(&k.fn, k.lib, k.name.c_str()));
    return E3_OK;
}

void jit_unload(JitKernel &k)
{
    if (k.lib) cudaLibraryUnload(k.lib);
    k.lib = nullptr;
    k.fn = nullptr;
}

}  // namespace e3
