"""Host-side guards (no GPU): the product never touches the oracle, the oracle never touches the product, nothing committed
reads the working folder, and the plumbing that ties bench.py's fp64 figures to an ncu capture behaves."""
import ast
import csv
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _imports(path):
    with open(path) as fh:
        tree = ast.parse(fh.read())
    names = set()
    for node in ast.walk(tree):
        if isinstance(node, ast.Import):
            names.update(a.name for a in node.names)
        elif isinstance(node, ast.ImportFrom) and node.module:
            names.add(node.module)
    return names


def test_product_and_oracle_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_2410_09146_b200")
    for f in os.listdir(pkg):
        if f.endswith(".py"):
            assert not any(n == "oracle" or n.startswith("oracle.") for n in _imports(os.path.join(pkg, f))), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert not any(n.startswith("paper_2410_09146_b200") for n in _imports(os.path.join(ROOT, "oracle", f))), f
    # the C++ / CUDA sources share no header either
    for f in ("phx_kernels.cu", "phx_device.cuh"):
        src = open(os.path.join(pkg, "csrc", f)).read()
        assert "orc" not in re.findall(r'#include\s+"([^"]+)"', src).__str__()
    assert "phx" not in re.findall(r'#include\s+"([^"]+)"', open(os.path.join(ROOT, "oracle", "orc.cpp")).read()).__str__()


def test_the_shared_input_module_holds_no_flux_or_inversion_code():
    """workloads.py is the only module both sides import: it may shape inputs, not evaluate the method."""
    src = open(os.path.join(ROOT, "paper_2410_09146_b200", "workloads.py")).read()
    for word in ("def prim_to_cons", "def cons_to_prim", "def riemann", "def hll", "def weno", "def recon", "def c2p", "ctypes", "import torch\n"):
        assert word not in src.split("def smooth_periodic_prims")[0], word


def test_nothing_committed_reads_the_working_folder():
    bad = []
    for base, dirs, files in os.walk(ROOT):
        dirs[:] = [d for d in dirs if d not in (".git", "_work", "gpurun_out", "__pycache__", ".pytest_cache", "baseline")]
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")) and f != "test_repo_rules.py":
                if "_work/" in open(os.path.join(base, f), errors="ignore").read():
                    bad.append(os.path.join(base, f))
    assert not bad, bad


def test_counts_file_is_tied_to_the_kernel_sources(tmp_path):
    from paper_2410_09146_b200 import profile_counts as pc
    path = os.path.join(ROOT, "profiles", "r02_kernel_counts.csv")
    rows, sha = pc.load(path, "cfg4_256")
    assert {"sweep_x", "sweep_y", "sweep_z", "update", "update_cfl"} <= set(rows)
    assert len(sha) == 16
    for k in ("sweep_x", "sweep_y", "sweep_z"):
        assert 600 < rows[k]["fp64_instr_per_zone"] < 900 and rows[k]["flop_per_zone"] > rows[k]["fp64_instr_per_zone"]
    # the committed capture is of the committed sources: bench.py will use it (a stale file makes it withhold the fp64 figures)
    assert sha == pc.source_hash(), "profiles/r02_kernel_counts.csv was captured from other kernel sources: re-capture"
    # a raw ncu export is reduced to one row per kernel class
    raw = tmp_path / "raw.csv"
    hdr = ["ID", "Kernel Name", "gpu__time_duration.sum", "launch__registers_per_thread", "smsp__cycles_elapsed.avg",
           "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum.per_cycle_elapsed", "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum.per_cycle_elapsed",
           "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum.per_cycle_elapsed", "dram__bytes_read.sum", "dram__bytes_write.sum",
           "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active"]
    units = ["", "", "ms", "register/thread", "cycle", "inst/cycle", "inst/cycle", "inst/cycle", "Gbyte", "Mbyte", "%", "%"]
    with open(raw, "w", newline="") as fh:
        w = csv.writer(fh)
        w.writerow(hdr); w.writerow(units)
        w.writerow(["0", "void k_sweep_march<0, 3, 1, 0>(MeshDev, const double *)", "1.0", "168", "1000", "10", "20", "30", "1.5", "500", "78", "18"])
        w.writerow(["1", "void k_sweep_march<0, 3, 1, 0>(MeshDev, const double *)", "3.0", "168", "1000", "10", "20", "30", "0.5", "500", "80", "18"])
        w.writerow(["2", "void k_update<0, 0, 1, 0, 0>(MeshDev)", "2.0", "72", "2000", "1", "1", "1", "4", "2000", "45", "42"])
    out = tmp_path / "counts.csv"
    import subprocess, sys
    subprocess.run([sys.executable, "-m", "paper_2410_09146_b200.profile_counts", str(raw), str(out), "--capture", "t", "--workload", "w", "--zones", "1000"],
                   check=True, cwd=ROOT)
    got, _ = pc.load(str(out), "w")
    assert got["sweep_y"]["launches"] == 2 and got["sweep_y"]["time_ms"] == 2.0
    assert got["sweep_y"]["fp64_instr_per_zone"] == 60.0 and got["sweep_y"]["flop_per_zone"] == 90.0      # (10+20+30) x 1000 cycles / 1000 zones
    assert got["sweep_y"]["dram_read_bytes"] == 1.0e9 and got["sweep_y"]["dram_write_bytes"] == 5.0e8
    assert got["update_cfl"]["registers"] == 72 and got["update_cfl"]["fp64_instr_per_zone"] == 6.0
