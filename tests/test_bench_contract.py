"""Host-side checks of bench.py (no GPU): the traffic table it reads for its `traffic` fields has the keys the roofline code
asks for, the peaks fall back when MEASURED_PEAKS.json is absent, and the reference arm (the oracle on a bounded sample, rank 0)
prints one JSON line with the contract's keys."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_traffic_table_has_the_keys_the_roofline_code_reads():
    import bench
    tr = bench.traffic_98k()
    # default path (chain kernel + B1) and the two-launch path (DHP_TC_FUSE=0)
    for key in ("nlist", "aev_fwd", "fused", "b1", "aev_bwd", "g1", "mid"):
        assert key in tr and tr[key] > 0, key
    # the chain kernel moves less DRAM than the two launches it replaced (the h1 round trip is gone)
    assert tr["fused"] < tr["g1"] + tr["mid"]


def test_peaks_have_the_three_denominators():
    import bench
    pk = bench.peaks()
    assert pk["hbm_gbs"] > 1000 and pk["bf16_tflops"] >= pk["bf16_tflops_sustained"] > 100
    assert pk["source"] in ("measured", "fallback")


def test_reference_arm_prints_the_contract_line():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "ani_energy_forces_atoms_evals_per_s" and d["unit"] == "atoms*evals/s"
    assert d["higher_is_better"] is True and d["value"] > 0 and d["steps"] == 1 and d["n_gpus"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
