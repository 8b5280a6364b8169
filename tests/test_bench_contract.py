"""bench.py on a box without a GPU: the reference arm prints the contract's JSON line, our arm refuses to run
(there is no CPU fallback to time).  CPU only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          cwd=ROOT, timeout=600)


def test_reference_arm_prints_the_contract_line():
    r = run_bench("--impl", "reference", "--steps", "2", "--warmup", "1", "--tracks", "600")
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "tracks/s" and line["higher_is_better"] is True
    assert line["steps"] == 2 and line["warmup"] == 1 and line["n_gpus"] == 1 and line["dtype"] == "f64"
    assert line["value"] > 0 and line["ms_per_step"] > 0 and line["vs_baseline"] is None
    assert line["config"]["workload"].startswith("cfg2") and line["config"]["tracks_per_step"] == 600
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == dict(value=line["value"], unit="tracks/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0)
    assert line["gpu_launches"] == 0


def test_reference_arm_under_torchrun_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, cwd=ROOT, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_our_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = run_bench("--steps", "1", "--warmup", "1", "--tracks", "100")
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def test_roofline_constants_are_the_numbers_of_the_committed_capture():
    """bench.py's executed-flop, FP64-pipe and DRAM-traffic constants (CAPTURE_COUNTS) are typed in from an ncu capture
    summarised under profiles/.  This re-reads that file -- the counter table's dram__bytes_* and FP64-pipe rows and the
    opcode table -- so that a refreshed capture and the constants cannot drift apart; and the hash that bench.py compares
    the built sources with must be the hash of csrc/ as committed (else the bench line reports the counts as null)."""
    import re
    sys.path.insert(0, ROOT)
    import bench
    cc = bench.CAPTURE_COUNTS
    txt = open(os.path.join(ROOT, cc["source"])).read()
    rows = {}
    for line in txt.splitlines():
        m = re.match(r"\| `([^`]+)` \| ([^|]*) \| (.*) \|$", line)
        if m and m.group(1) not in rows:
            rows[m.group(1)] = (m.group(2).strip(), [c.strip() for c in m.group(3).split(" | ")])
    kernels = rows["Kernel Name"][1]
    col = {k: [i for i, n in enumerate(kernels) if k in n][0] for k in ("kf_forward_kernel", "kf_rts_kernel")}
    for k, i in col.items():
        assert rows["dram__bytes_read.sum"][0] == "Gbyte" and rows["dram__bytes_write.sum"][0] == "Gbyte"
        got = (float(rows["dram__bytes_read.sum"][1][i]), float(rows["dram__bytes_write.sum"][1][i]))
        assert got == pytest.approx(cc["dram_gbyte"][k], rel=1e-6), (k, got)
        pct = float(rows["sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"][1][i])
        assert abs(pct - cc["fp64_pipe_pct"][k]) < 0.06, (k, pct)
        # opcode table: "    void kf::<kernel><...>: ..." followed by "      DFMA    172.182 M ..."
        blk = txt[txt.index("void kf::" + k):]
        blk = blk[:blk.index("\n\n")]
        for op, want in cc["opcodes_M"][k].items():
            m = re.search(r"^\s+%s\s+([0-9.]+) M" % op, blk, flags=re.M)
            assert m and float(m.group(1)) == pytest.approx(want, abs=5e-4), (k, op, m and m.group(1))
    # the derived per-leg figures are those of the opcode counts (DFMA = 2 flop)
    f = cc["opcodes_M"]["kf_forward_kernel"]
    assert bench.EXECUTED_PER_LEG["flop"]["kf_forward_kernel"] == pytest.approx(
        (2 * f["DFMA"] + f["DMUL"] + f["DADD"]) * 1e6 * 32 / (262144 * 30))
    assert 1800 < bench.EXECUTED_PER_LEG["flop"]["kf_forward_kernel"] < 1830
    assert bench.NCU_TRAFFIC["bytes_per_leg"]["kf_rts_kernel"] == pytest.approx(441.0, rel=0.02)
    assert bench.CAPTURE["sources_sha16"] == bench.kernel_sources_sha16(), \
        "csrc/ changed since the capture bench.py's roofline constants come from: refresh " + cc["source"]
