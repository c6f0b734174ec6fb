"""TEST INFRASTRUCTURE (tests/emu/README.md): paper_2606_07759_b200/csrc/*.cu -> host C++ for the emulation.

The kernels' own source is kept line for line; only what cannot exist on a host is rewritten: ``k<<<grid, block, smem,
stream>>>(args)`` becomes ``EMU_LAUNCH``, ``__shared__`` becomes ``static`` (one CTA runs at a time), the dynamic
shared-memory array becomes the emulator's arena, and the bodies of the one-line inline-PTX helpers (mbarrier, TMA,
ld/st.shared, cp.async, bar.sync, the cache-hinted weight load) and the predicated-load block of the sampler get C
equivalents that go through the emulator's bounds checks."""
import os
import re
import shutil

SRC = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "..", "paper_2606_07759_b200", "csrc")

BODIES = {
    "mbar_init": "{ emu::mbar_init(bar, count); }",
    "fence_barrier_init": "{ }",
    "fence_proxy_async": "{ }",
    "mbar_expect_tx": "{ emu::mbar_arrive_expect_tx(bar, bytes); }",
    "mbar_try_wait": "{ return emu::mbar_try_wait(bar, parity); }",
    "tma_load_box": "{ emu::mbar_complete_tx(bar, emu_tma(dst, map, x, y, z)); }",
    "tma_load_box_plain": "{ emu::mbar_complete_tx(bar, emu_tma(dst, map, x, y, z)); }",
    "lds_f32": '{ return *(float *)emu::shared_ptr(addr, 4, "lds_f32"); }',
    "lds_s32": '{ return *(int *)emu::shared_ptr(addr, 4, "lds_s32"); }',
    "sts_f32": '{ *(float *)emu::shared_ptr(addr, 4, "sts_f32") = v; }',
    "sts_s32": '{ *(int *)emu::shared_ptr(addr, 4, "sts_s32") = v; }',
    "red_shared_f32": '{ *(float *)emu::shared_ptr(addr, 4, "red_shared_f32") += v; }',
    "cp_async_4": '{ emu::check_global(src, 4, "cp_async_4"); memcpy(emu::shared_ptr(dst, 4, "cp_async_4"), src, 4); }',
    "cp_async_wait_all": "{ }",
    "bar_sync": "{ (void)id; (void)nthreads; emu::cta_barrier(); }",
    "wld": '{ emu::check_global(p, 4, "wld"); return *p; }',
}
TMA = r'''
static inline uint32_t emu_tma(void *dst, const void *map, int x, int y, int z)   // -> bytes delivered
{
    EmuTensorMap m; memcpy(&m, map, sizeof(m));
    const uint32_t a = emu::shared_addr(dst);
    if (a % 128) emu::fail("TMA destination is not 128-byte aligned");
    float *d = (float *)emu::shared_ptr(a, 4, "tma") ;
    emu::shared_ptr(a + (m.box[0] * m.box[1] * m.box[2] - 1) * 4u, 4, "tma (end of box)");
    if (m.box[2] != 1) emu::fail("TMA box depth");
    for (uint32_t r = 0; r < m.box[1]; ++r)
        for (uint32_t c = 0; c < m.box[0]; ++c) {
            const long long X = (long long)x + c, Y = (long long)y + r, Z = z;
            float v = 0.0f;
            if (X >= 0 && X < (long long)m.dims[0] && Y >= 0 && Y < (long long)m.dims[1] && Z >= 0 && Z < (long long)m.dims[2]) {
                const float *src = (const float *)((const char *)m.base + Z * (long long)m.strides[1] + Y * (long long)m.strides[0]) + X;
                emu::check_global(src, 4, "tma source");
                v = *src;
            }
            d[r * m.box[0] + c] = v;
        }
    return m.box[0] * m.box[1] * m.box[2] * 4u;
}
'''

def replace_body(s, name):
    m = re.search(r"__device__ __forceinline__ [\w ]+\b%s\(" % name, s)
    if not m:
        return s
    i = s.index("{", s.index(")", m.end()))
    depth, j = 0, i
    while True:
        if s[j] == "{": depth += 1
        elif s[j] == "}":
            depth -= 1
            if depth == 0: break
        j += 1
    return s[:i] + BODIES[name] + s[j + 1:]

def convert(name, out_dir):
    s = open(os.path.join(SRC, name)).read()
    for n in BODIES:
        s = replace_body(s, n)
    # the predicated-load block of sample()
    a = s.find("        float phi;\n        asm volatile(")
    if a >= 0:
        b = s.index("        return phi;", a)
        s = s[:a] + '''        float phi = 0.0f;
        if (__float_as_uint(col) < cw_bits && __float_as_uint(row) < ch_bits) {
            const float v00 = lds_f32(at), v01 = lds_f32(at + 4u), v10 = lds_f32(at + rpitch4), v11 = lds_f32(at + rpitch4 + 4u);
            const float t = fmaf(fx, v01 - v00, v00), u = fmaf(fx, v11 - v10, v10);
            phi = fmaf(fy, u - t, t);
        }
''' + s[b:]
    s = s.replace("extern __shared__ __align__(128) float patch[];", "float *patch = (float *)emu::smem;")
    s = re.sub(r"\b__shared__\b", "static", s)
    # launches
    def launch(m):
        return "EMU_LAUNCH(%s, %s, %s);" % (m.group(1), m.group(2), m.group(3))
    s = re.sub(r"(\w+)<<<(.*?)>>>\((.*?)\);", lambda m: "{ auto cfg_ = std::make_tuple(%s); EMU_LAUNCH(%s, std::get<0>(cfg_), std::get<1>(cfg_), std::get<2>(cfg_), %s); }" % (m.group(2), m.group(1), m.group(3)), s, flags=re.S)
    s = s.replace('#include "synim_device.h"', '#include "synim_device.h"\n#include <tuple>\n#include <cuda.h>\n' + (TMA if name == "synim_strip.cu" else ""), 1)
    open(os.path.join(out_dir, name.replace(".cu", ".cpp")), "w").write(s)

SOURCES = ("synim_api.cu", "synim_kernels.cu", "synim_strip.cu", "synim_popt.cu")


def convert_all(out_dir):
    os.makedirs(out_dir, exist_ok=True)
    for n in SOURCES:
        convert(n, out_dir)
    shutil.copy(os.path.join(SRC, "synim_device.h"), os.path.join(out_dir, "synim_device.h"))
    return [os.path.join(out_dir, n.replace(".cu", ".cpp")) for n in SOURCES]
