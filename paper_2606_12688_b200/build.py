"""Build ``libmstar_attn.so`` (and the bench-only ``bench_aux/libmstar_benchaux.so``) in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_12688_b200.build [--force] [--verbose]
    python -m paper_2606_12688_b200.build --sass-counts      # per-kernel counts of the Blackwell SASS mnemonics (markdown)

The shared library travels to the GPU box with the repo snapshot; nothing is JIT-compiled there.
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
LIB_PATH = os.path.join(PKG_DIR, "libmstar_attn.so")
SOURCES = ["host_common.cu", "kv_append.cu", "kv_append_fp8.cu", "kv_transfer.cu", "decode.cu", "merge_states.cu",
           "prefill.cu", "prefill_umma.cu", "prefill_fp8.cu", "sampling.cu"]
# measurement aid for bench.py, a library of its own (not part of the product ABI)
AUX_DIR = os.path.join(PKG_DIR, "bench_aux")
AUX_LIB_PATH = os.path.join(AUX_DIR, "libmstar_benchaux.so")
AUX_SOURCES = ["hbm_probe.cu"]
HEADERS = ["host_common.h", "ptx.cuh", "umma.cuh", os.path.join("..", "..", "include", "mstar_attn.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB_PATH) or not os.path.exists(AUX_LIB_PATH):
        return True
    t = min(os.path.getmtime(LIB_PATH), os.path.getmtime(AUX_LIB_PATH))
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(AUX_DIR, f) for f in AUX_SOURCES]
    deps.append(os.path.abspath(__file__))
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB_PATH
    objs = []
    procs = []
    build_dir = os.path.join(PKG_DIR, "build")
    os.makedirs(build_dir, exist_ok=True)
    aux_objs = []
    for src_dir, src in [(CSRC, f) for f in SOURCES] + [(AUX_DIR, f) for f in AUX_SOURCES]:
        obj = os.path.join(build_dir, src.replace(".cu", ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, "-c", os.path.join(src_dir, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
            print(" ".join(cmd), flush=True)
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        (objs if src_dir == CSRC else aux_objs).append(obj)
    failed = False
    for src, pr in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0:
            failed = True
            sys.stderr.write("nvcc failed on %s:\n%s\n" % (src, out))
        elif verbose or out.strip():
            sys.stderr.write(out)
    if failed:
        raise RuntimeError("nvcc failed; see messages above")
    for path, parts in ((LIB_PATH, objs), (AUX_LIB_PATH, aux_objs)):
        tmp = path + ".tmp.%d" % os.getpid()
        link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *parts, "-cudart",
                "static"]
        subprocess.check_call(link)
        os.replace(tmp, path)
    return LIB_PATH


SASS_MNEMONICS = ["UTCHMMA", "UTCQMMA", "LDTM", "STTM", "UTMALDG", "UTMASTG", "UBLKCP", "UTCBAR", "HMMA", "LDSM",
                  "MUFU.EX2", "SYNCS", "STL", "LDL"]


def sass_counts() -> str:
    """Markdown table: how often each mnemonic of interest occurs in every kernel of the built library
    (`cuobjdump -sass`; the evidence table of B200_PROFILING.md: tcgen05.mma = UTC*MMA, tcgen05.ld/st = LDTM/STTM,
    TMA = UTMALDG/UTMASTG/UBLKCP, mma.sync = HMMA; STL/LDL = register spills)."""
    import re
    build_library()
    cuobjdump = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "cuobjdump")
    out = subprocess.run([cuobjdump, "-sass", LIB_PATH], capture_output=True, text=True, check=True).stdout
    demangle = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "cu++filt")
    rows, name, counts = [], None, None
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            if name:
                rows.append((name, counts))
            name, counts = m.group(1), dict.fromkeys(SASS_MNEMONICS, 0)
            continue
        if name and re.match(r"\s+/\*[0-9a-f]{4,}\*/", line):
            body = line.split("*/", 1)[1]
            for mn in SASS_MNEMONICS:
                if re.search(r"(?<![A-Z0-9_.])" + re.escape(mn) + r"(?![A-Z0-9_])", body):
                    counts[mn] += 1
    if name:
        rows.append((name, counts))
    names = subprocess.run([demangle] + [r[0] for r in rows], capture_output=True, text=True).stdout.splitlines()
    lines = ["| kernel | " + " | ".join(SASS_MNEMONICS) + " |", "|---|" + "---|" * len(SASS_MNEMONICS)]
    for (_, c), nm in sorted(zip(rows, names), key=lambda x: x[1]):
        short = nm[:nm.index(">(") + 1] if ">(" in nm else nm.split("(")[0]
        short = short.replace("mstar::", "").replace("void ", "").replace("(int)", "").replace("(bool)", "")
        lines.append("| `%s` | " % short + " | ".join(str(c[m]) for m in SASS_MNEMONICS) + " |")
    return "\n".join(lines)


if __name__ == "__main__":
    if "--sass-counts" in sys.argv:
        print(sass_counts())
    else:
        print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
