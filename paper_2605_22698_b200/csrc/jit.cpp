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

int jit_compile(JitKernel &k, const std::string &file_hint)
{
    // keep the generated source on disk so that -lineinfo maps SASS back to it (ncu source page)
    std::string dir = "/tmp/e3b200_jit";
    mkdir(dir.c_str(), 0777);
    size_t h = std::hash<std::string>{}(k.source);
    char hb[32];
    snprintf(hb, sizeof(hb), "%016zx", h);
    std::string path = file_hint.empty() ? dir + "/" + k.name + "_" + hb + ".cu" : file_hint;
    if (FILE *f = fopen(path.c_str(), "w")) { fwrite(k.source.data(), 1, k.source.size(), f); fclose(f); }

    // compiled-code cache (speed only: the key is the hash of the generated source plus the NVRTC version; E3_JIT_CACHE=0 disables it)
    int vmaj = 0, vmin = 0;
    nvrtcVersion(&vmaj, &vmin);
    char vb[64];
    snprintf(vb, sizeof(vb), "_%zu_nvrtc%d_%d", k.source.size(), vmaj, vmin);
    const char *cache_env = getenv("E3_JIT_CACHE");
    const bool use_cache = !(cache_env && cache_env[0] == '0') && file_hint.empty();
    const std::string cpath = dir + "/" + k.name + "_" + hb + vb + ".cubin", ipath = cpath + ".info";
    if (use_cache) {
        FILE *fi = fopen(ipath.c_str(), "r"), *fc = fopen(cpath.c_str(), "rb");
        long long want = -1;
        int regs = 0, spill = 0, smem = 0;
        if (fi && fc && fscanf(fi, "%lld %d %d %d", &want, &regs, &spill, &smem) == 4 && want > 0) {
            k.cubin.resize((size_t)want);
            if (fread(k.cubin.data(), 1, (size_t)want, fc) == (size_t)want && fgetc(fc) == EOF) {
                fclose(fi); fclose(fc);
                k.regs = regs; k.spill = spill; k.smem = smem;
                return E3_OK;
            }
            k.cubin.clear();
        }
        if (fi) fclose(fi);
        if (fc) fclose(fc);
    }

    nvrtcProgram prog;
    if (nvrtcCreateProgram(&prog, k.source.c_str(), path.c_str(), 0, nullptr, nullptr) != NVRTC_SUCCESS) {
        set_error("nvrtcCreateProgram failed");
        return E3_ERR_JIT;
    }
    const char *cuda_home = getenv("CUDA_HOME");
    std::string inc = std::string("-I") + (cuda_home ? cuda_home : "/usr/local/cuda") + "/include";
    const char *opts[] = { "--gpu-architecture=sm_100a", "-lineinfo", "--std=c++17", "--ptxas-options=-v",
                           "-default-device", inc.c_str() };
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
                  fprintf(fi, "%lld %d %d %d\n", (long long)k.cubin.size(), k.regs, k.spill, k.smem) > 0;
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
