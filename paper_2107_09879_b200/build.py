"""Builds paper_2107_09879_b200/libtm.so (the C-ABI CUDA library, include/tm.h) in-tree (lib/libtm.so) with nvcc for sm_100a.

    python -m paper_2107_09879_b200.build [--force] [-v]

nvcc cross-compiles without a GPU; the translation units (host code + one per kernel family) compile in parallel.  The generated headers under csrc/generated/ are (re)written by
csrc/gen_tables.py when missing or older than the generator.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated")
SO = os.path.join(HERE, "lib", "libtm.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _mtime(p):
    return os.path.getmtime(p) if os.path.exists(p) else 0.0


def _gen_hash():
    import hashlib
    return hashlib.sha256(open(os.path.join(CSRC, "gen_tables.py"), "rb").read()).hexdigest()


def generate(force=False):
    """(Re)write csrc/generated/ when it does not belong to the current gen_tables.py.  Staleness is decided by the
    generator's content hash recorded in generated/GENERATOR_SHA256 (file times mean nothing after a git checkout, and a
    full generation takes minutes of 40-digit arithmetic)."""
    gen_py = os.path.join(CSRC, "gen_tables.py")
    stamp = os.path.join(GEN, "GENERATOR_SHA256")
    outs = [os.path.join(GEN, f) for f in ("tm_tables_gen.h", "tm_coplanar_gen.cuh", "tm_coplanar_f2_gen.cuh",
                                           "tm_general3d_gen.cuh", "tm_coplanar4_gen.cuh", "tm_rot3d_gen.cuh", "tm_rot3d_ws_gen.cuh")]
    have = open(stamp).read().strip() if os.path.exists(stamp) else ""
    if force or have != _gen_hash() or not all(os.path.exists(o) for o in outs):
        subprocess.check_call([sys.executable, gen_py])
        with open(stamp, "w") as f:
            f.write(_gen_hash() + "\n")


def sources():
    out = [os.path.join(HERE, "..", "include", "tm.h")]
    for root, _, files in os.walk(CSRC):
        out += [os.path.join(root, f) for f in files if f.endswith((".cu", ".cuh", ".h"))]
    return out


# Translation units: the host code and one per all-pairs kernel family (the generated straight-line code makes ptxas the
# long pole of the build - compiled in parallel, the wall time is that of the largest family instead of their sum).
UNITS = ["tm_api.cu", "tm_tu_coplanar.cu", "tm_tu_cop4_lo.cu", "tm_tu_cop4_hi.cu", "tm_tu_sym3d.cu", "tm_tu_rot3d_lo.cu",
         "tm_tu_rot3d_6.cu", "tm_tu_rot3d_7.cu", "tm_tu_general.cu", "tm_tu_rot3d_ws.cu", "tm_static.cu"]
CFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def build(force=False, verbose=False, jobs=None):
    generate()
    if not force and _mtime(SO) >= max(_mtime(s) for s in sources()):
        return SO
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(os.path.dirname(SO), exist_ok=True)
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    extra = os.environ.get("TM_NVCC_EXTRA", "").split()             # e.g. -DTM_COP4_SYNC_L6=255 for A/B builds

    flag_file = os.path.join(objdir, "FLAGS")
    flags_now = " ".join(CFLAGS + extra)
    same_flags = os.path.exists(flag_file) and open(flag_file).read() == flags_now

    def up_to_date(obj, dep):
        """obj is newer than every file nvcc listed as a dependency of the unit (make-style .d file)."""
        if force or verbose or not same_flags or not (os.path.exists(obj) and os.path.exists(dep)):
            return False
        words = open(dep).read().replace("\\\n", " ").split()
        return all(os.path.exists(f) and _mtime(f) <= _mtime(obj) for f in words[1:] if not f.endswith(":"))

    def compile_one(unit):
        obj = os.path.join(objdir, unit[:-3] + ".o")
        dep = obj + ".d"
        if up_to_date(obj, dep):
            return unit, obj, subprocess.CompletedProcess([], 0, "", "")
        cmd = ([NVCC] + CFLAGS + extra + (["-Xptxas", "-v"] if verbose else [])
               + ["-MD", "-MF", dep, "-c", "-o", obj, os.path.join(CSRC, unit)])
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        return unit, obj, r
    with ThreadPoolExecutor(max_workers=jobs or min(len(UNITS), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, UNITS))
    for unit, obj, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(f"== {unit}\n{r.stdout}{r.stderr}")
        if r.returncode != 0:
            raise subprocess.CalledProcessError(r.returncode, f"nvcc -c {unit}")
    with open(flag_file, "w") as f:
        f.write(flags_now)
    subprocess.check_call([NVCC, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", SO]
                          + [obj for _, obj, _ in results], cwd=CSRC)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
