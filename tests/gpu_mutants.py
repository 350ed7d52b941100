"""Sensitivity check of the GPU parity suite (run by hand; not collected by pytest): one-token mistakes in the CUDA kernels
— the same kind the oracle's mutation harness injects into oracle/ocn_ref.cpp — must make `pytest -m gpu` parity tests fail.

    python tests/gpu_mutants.py --build DIR      # here or on the box: builds one libocn per mutant into DIR (nvcc, parallel)
    python tests/gpu_mutants.py --run DIR        # on a B200: swaps each library in, runs the parity tests, restores the original

The mutants are applied to scratch copies of paper_2309_06662_b200/csrc; the tree is not modified.  Result table: DESIGN.md §5.1.
"""
import argparse
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2309_06662_b200", "csrc")
SO = os.path.join(ROOT, "paper_2309_06662_b200", "libocn.so")
TESTS = ["tests/test_gpu_parity.py", "tests/test_gpu_closure.py", "tests/test_gpu_variants.py", "tests/test_gpu_forcing.py"]

# (name, file in csrc, exact text (once), replacement)
MUTANTS = [
    ("k1_coriolis_north_half", "kernels_tile.cuh",
     "X(fFn) * half * X(dxFn) * vsum_n), dxCj, rdxCj);", "X(fFj) * half * X(dxFn) * vsum_n), dxCj, rdxCj);"),
    ("k1_w_sign", "kernels_tile.cuh",
     "wa = (X(wa) - X((double)dzk) * X((double)Dc)).v;", "wa = (X(wa) + X((double)dzk) * X((double)Dc)).v;"),
    ("k1_south_face_length", "kernels_tile.cuh",
     "const T len = isy ? s_dxF[row] : dy;", "const T len = isy ? s_dxC[row] : dy;"),
    ("k1_ab2_sign_u", "kernels_tile.cuh",
     "const T Ghu = (X(c0) * X(Gu) - X(c1) * X(gm_u)).v;", "const T Ghu = (X(c0) * X(Gu) + X(c1) * X(gm_u)).v;"),
    ("k1_vertical_advection_v_area", "kernels_tile.cuh",
     "const T volf = (X(AzFj) * X(dzk)).v;", "const T volf = (X(AzCj) * X(dzk)).v;"),
    ("strip_u_metric", "kernels_column.cuh",
     "cu[r] = dtau * g * P.Hu[c] * rdxr; gu[r] = dtau * P.GU[c];", "cu[r] = dtau * g * P.Hu[c] * rdy; gu[r] = dtau * P.GU[c];"),
    ("tile_eta_metric_fp64", "kernels_column.cuh",
     "X(dF[y + 1]) * X(sV[q + EX]) - X(dF[y]) * X(sV[q])),", "X(dF[y]) * X(sV[q + EX]) - X(dF[y]) * X(sV[q])),"),
    ("k3_correction_depth", "kernels_column.cuh",
     "const T cu = tx1 < nz ? (P.Ub[c] - P.SU[c]) * P.rHu[c] : T(0);", "const T cu = tx1 < nz ? (P.Ub[c] - P.SU[c]) * P.rHv[c] : T(0);"),
    ("pressure_trapezoid_spacing", "kernels_column.cuh",
     ": E::sub(p_above, E::mul(E::mul(0.5, E::add(b1, b0)), P.dzc_d[k + 1]));",
     ": E::sub(p_above, E::mul(E::mul(0.5, E::add(b1, b0)), P.dzc_d[k]));"),
    ("closure_nu_power_fp32", "kernels_mixing.cuh",
     "const float g2 = R.nu0 * f * f;\n    return make_float2(R.nuz + g2 + conv, R.kapz + g2 * f + conv);",
     "const float g2 = R.nu0 * f;\n    return make_float2(R.nuz + g2 + conv, R.kapz + g2 * f + conv);"),
    ("weno5_pair_linear_weight", "common.cuh",
     "a1 = mul2(mul2(f2(0.6f), b02), b02);", "a1 = mul2(mul2(f2(0.5f), b02), b02);"),
    ("strip_transport_filter_weight", "kernels_column.cuh",
     "for (int r = 0; r < 4; ++r) { be[r] += am * e[r]; bU[r] += bm * u[r]; bV[r] += bm * v[r]; }",
     "for (int r = 0; r < 4; ++r) { be[r] += am * e[r]; bU[r] += am * u[r]; bV[r] += bm * v[r]; }"),
    ("k1_restoring_sign", "kernels_tile.cuh",
     "X(P.gamma_T) * (X(rtg.x) - X(tsc.x))", "X(P.gamma_T) * (X(tsc.x) - X(rtg.x))"),
    ("k1_drag_speed_u", "kernels_tile.cuh",
     "X(P.drag_cd) * X((T)sqrt((X(u_c) * X(u_c) + X(vhat) * X(vhat)).v))) * X(u_c), dzk, rdzk)",
     "X(P.drag_cd) * X((T)sqrt((X(u_c) * X(u_c)).v))) * X(u_c), dzk, rdzk)"),
    ("eos_cabbeling_power", "kernels_column.cuh",
     "E::add(E::mul(P.ath_d[k], dT), E::mul(E::mul(P.ha2_d, dT), dT))", "E::add(E::mul(P.ath_d[k], dT), E::mul(P.ha2_d, dT))"),
    ("biharmonic_divergence_row", "kernels_biharmonic.cuh",
     "const Xv<T> Ds = xdiv(X(dy) * (X(vse.x) - X(vs.x)) + X(dxFj) * X(v00.y) - X(dxFs) * X(vs.y), AzCs, rAzCs);",
     "const Xv<T> Ds = xdiv(X(dy) * (X(vse.x) - X(vs.x)) + X(dxFj) * X(v00.y) - X(dxFs) * X(vs.y), AzCj, rAzCj);"),
]


def build(outdir):
    os.makedirs(outdir, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC", "-shared"]

    def one(m):
        name, fname, old, new = m
        tmp = tempfile.mkdtemp(prefix="ocn_gpumut_")
        try:
            pkg = os.path.join(tmp, "paper_2309_06662_b200")
            shutil.copytree(CSRC, os.path.join(pkg, "csrc"))
            shutil.copytree(os.path.join(ROOT, "include"), os.path.join(tmp, "include"))
            path = os.path.join(pkg, "csrc", fname)
            text = open(path).read()
            assert text.count(old) == 1, "mutation target not found exactly once: " + name
            open(path, "w").write(text.replace(old, new))
            subprocess.check_call([nvcc] + flags + ["-o", os.path.join(outdir, "libocn_%s.so" % name), os.path.join(pkg, "csrc", "ocn_api.cu")])
        finally:
            shutil.rmtree(tmp, ignore_errors=True)
        return name

    with ThreadPoolExecutor(max_workers=max(1, (os.cpu_count() or 4) // 2)) as ex:
        for name in ex.map(one, MUTANTS):
            print("built", name, flush=True)


def run(indir):
    keep = SO + ".keep"
    shutil.copy2(SO, keep)
    rows = []
    try:
        for name, fname, _, _ in MUTANTS:
            lib = os.path.join(indir, "libocn_%s.so" % name)
            shutil.copy(lib, SO)
            os.utime(SO, None)                                   # newer than the sources: build.build() leaves it alone
            r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider"] + TESTS, cwd=ROOT,
                               stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            first = [ln for ln in r.stdout.splitlines() if ln.startswith("FAILED")]
            rows.append((name, fname, r.returncode, first[0][:150] if first else ("SURVIVES" if r.returncode == 0 else "rc=%d" % r.returncode)))
            print("%-32s %-22s %s" % (name, fname, rows[-1][3]), flush=True)
    finally:
        shutil.copy2(keep, SO)
        os.utime(SO, None)
        os.remove(keep)
    print("survivors:", [r[0] for r in rows if r[2] == 0])


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--build")
    ap.add_argument("--run")
    ap.add_argument("--only", default="", help="comma-separated mutant names (default: all)")
    a = ap.parse_args()
    if a.only:
        MUTANTS[:] = [m for m in MUTANTS if m[0] in a.only.split(",")]
    if a.build:
        build(a.build)
    if a.run:
        run(a.run)
