"""Build libckb.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1309_2710_b200.build [--force] [--verbose]

One object per kernel instantiation (csrc/ckb_inst.cu compiled with -DCKB_L/-DCKB_NV, the list is read
from CKB_FOR_THREAD / CKB_FOR_GROUP in csrc/ckb_host.h), compiled in parallel, then linked together
with the API and probe objects.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import hashlib
import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libckb.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", OBJ, *ARCH]


def instantiations():
    txt = open(os.path.join(CSRC, "ckb_host.h")).read()
    out = []
    for name in ("CKB_FOR_THREAD", "CKB_FOR_GROUP"):
        line = re.search(r"#define %s\(X\)(.*)" % name, txt).group(1)
        out += [(int(a), int(b)) for a, b in re.findall(r"X\((\d+),\s*(\d+)\)", line)]
    return out


def min_blocks(L: int, NV: int, method: str = "rkck") -> int:
    """Resident 128-thread blocks per SM that the register allocation of integrate_kernel<L, NV> must allow
    (launch bounds): 4 -> <= 128 registers, 3 -> <= 168, 2 -> <= 255.  Chosen so that no instantiation spills."""
    if L == 1:  # thread-per-ODE: k3..k5 (RKCK) / v (RKC) sit in shared scratch so that 3 blocks fit
        if method == "rkc":
            return 2
        return 3 if NV <= 14 else 2
    if L in (2, 4):  # few lanes per system: small mechanisms, short stage vectors
        return 4 if NV <= 5 else 3
    if NV <= 2:  # register slots per stage vector
        return 4
    if NV <= 4:
        return 3
    return 2


def tmem_tables(L: int, NV: int) -> int:
    """1 = the object also carries warp-per-ODE integrate kernels that read the reaction-slot table from tensor memory
    (tcgen05.ld) instead of global memory / L1: one block of 512 threads per SM then owns the SM's
    512 TMEM columns, sized by tmem_block()."""
    return 1 if (L == 32 and NV in (2, 4)) else 0


def tmem_block(L: int, NV: int) -> int:
    """Threads of the one block per SM of the TMEM kernels: what the registers allow (128 per thread for NV = 2, 168
    for NV = 4, the 111-species class)."""
    return 512 if NV <= 2 else 384


def exp_table_flags(L: int):
    """Warp-per-ODE objects: exp through a 64-entry table of 2^(j/64) in shared memory, 16 copies so that every lane reads
    its own bank pair (12 instead of 17 FP64 instructions per exponential, dependency chain 9 instead of 14): configs[3]
    168.8k -> 173.6k ODE/s.  The narrower mappings keep the polynomial (their shared-memory pipe is the busier unit)."""
    return ["-DCKB_EXP_TABLE=1", "-DCKB_EXP_TABLE_REPL=16"] if L == 32 else []


def block_threads(L: int, NV: int) -> int:
    """Threads per block of the table-driven kernels (CKB_BLOCK)."""
    return 128


def _digest(extra: str) -> str:
    h = hashlib.sha256(extra.encode())
    h.update(open(os.path.abspath(__file__), "rb").read())  # the per-instantiation knobs live in this file
    for root in (CSRC, os.path.join(HERE, "..", "include")):
        for fn in sorted(os.listdir(root)):
            if fn.endswith((".cu", ".cuh", ".h")):
                h.update(fn.encode())
                h.update(open(os.path.join(root, fn), "rb").read())
    return h.hexdigest()


def _embed_sources():
    """The device headers as string literals (build/ckb_embed.inc): ckb_gen.cu hands them to the runtime compiler."""
    out = []
    for var, fn in (("ckb_embed_tables", "ckb_tables.h"), ("ckb_embed_device", "ckb_device.cuh")):
        txt = open(os.path.join(CSRC, fn)).read()
        assert ')CKBSRC"' not in txt
        # string literals are limited to 64 KiB by some compilers: concatenate raw-string chunks cut at line ends
        chunks, cur = [], ""
        for line in txt.splitlines(keepends=True):
            if len(cur) + len(line) > 12000:
                chunks.append(cur)
                cur = ""
            cur += line
        chunks.append(cur)
        out.append("static const char %s[] =\n%s;\n" % (var, "\n".join('R"CKBSRC(%s)CKBSRC"' % c for c in chunks)))
    path = os.path.join(OBJ, "ckb_embed.inc")
    new = "".join(out)
    if not os.path.exists(path) or open(path).read() != new:
        with open(path, "w") as fh:
            fh.write(new)


def _run(cmd, verbose):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    if verbose:
        sys.stderr.write(r.stdout + r.stderr)


def build(force: bool = False, verbose: bool = False, ptxas_v: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    flags = FLAGS + (["-Xptxas", "-v"] if ptxas_v else [])
    stamp = os.path.join(OBJ, "stamp")
    digest = _digest(" ".join(flags))
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == digest:
        return LIB
    _embed_sources()
    jobs = []
    for src in ("ckb_api.cu", "ckb_pack.cu", "ckb_order.cu", "ckb_probe.cu", "ckb_gen.cu", "ckb_thread.cu", "ckb_chemkin.cu"):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        jobs.append((obj, [NVCC, *flags, "-c", os.path.join(CSRC, src), "-o", obj]))
    for (L, NV) in instantiations():
        obj = os.path.join(OBJ, f"ckb_inst_L{L}_NV{NV}.o")
        bt = block_threads(L, NV)
        jobs.append((obj, [NVCC, *flags, f"-DCKB_L={L}", f"-DCKB_NV={NV}", f"-DCKB_BLOCK={bt}",
                           f"-DCKB_MINB={max(1, min_blocks(L, NV) * 128 // bt)}", f"-DCKB_MINB_RKC={max(1, min_blocks(L, NV, 'rkc') * 128 // bt)}",
                           f"-DCKB_TMEM={tmem_tables(L, NV)}", f"-DCKB_TMEM_BLOCK={tmem_block(L, NV)}",
                           f"-DCKB_TMEM_MIN_N={148 * tmem_block(L, NV) // 32}",
                           *exp_table_flags(L),
                           "-c",
                           os.path.join(CSRC, "ckb_inst.cu"), "-o", obj]))
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        list(ex.map(lambda j: _run(j[1], verbose or ptxas_v), jobs))
    tmp = LIB + f".tmp{os.getpid()}"
    _run([NVCC, "-shared", *ARCH, "-o", tmp, *[j[0] for j in jobs], "-ldl"], verbose)
    os.replace(tmp, LIB)
    with open(stamp, "w") as fh:
        fh.write(digest)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, ptxas_v="--ptxas-v" in sys.argv))
