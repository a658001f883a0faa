"""paper_1902_03252_b200/ncu_extract.py on a hand-written export in the layout of `ncu --page raw --csv --print-units base`:
the longest launch of the named kernel is taken, its DRAM bytes land in the JSON under workload/mode with the commit, the
markdown table carries the counters with their units."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CSV = '''==PROF== Connected to process 1
"ID","Kernel Name","gpu__time_duration.sum","dram__bytes_read.sum","dram__bytes_write.sum","launch__registers_per_thread"
"","","ns","byte","byte","register/thread"
"0","void lt_grad_f64_kernel<LtDpieModel, 1, 4>(const double *)","500","10","20","54"
"1","void lt_grad_f64_kernel<LtDpieModel, 4, 2>(const double *)","68,000,000","104,857","268435456","126"
"2","lt_flag_kernel(const float2 *)","70","1","2","58"
'''


def test_extract_json_and_markdown(tmp_path):
    js, md = tmp_path / "t.json", tmp_path / "t.md"
    r = subprocess.run([sys.executable, "-m", "paper_1902_03252_b200.ncu_extract", "--kernel", "lt_grad_f64_kernel",
                        "--workload", "cfg3_4096x4096_1000", "--mode", "fp64", "--commit", "abc1234", "--json", str(js),
                        "--md", str(md)], input=CSV, capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    rec = json.load(open(js))
    e = rec["captures"]["cfg3_4096x4096_1000/fp64"]
    assert rec["commit"] == "abc1234" and e["launches_in_report"] == 2 and "4, 2" in e["kernel"]
    assert e["dram_bytes_read"] == 104857 and e["dram_bytes_write"] == 268435456
    text = open(md).read()
    assert "| `launch__registers_per_thread` | register/thread | 126 |" in text and "lt_flag_kernel" not in text
    # a second capture is merged into the same file
    r = subprocess.run([sys.executable, "-m", "paper_1902_03252_b200.ncu_extract", "--kernel", "lt_flag_kernel",
                        "--workload", "w", "--mode", "mixed", "--json", str(js)], input=CSV, capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0 and set(json.load(open(js))["captures"]) == {"cfg3_4096x4096_1000/fp64", "w/mixed"}
    # --sum: the launches of one step (a catalogue beyond one constant-bank slot-load) are added up
    r = subprocess.run([sys.executable, "-m", "paper_1902_03252_b200.ncu_extract", "--sum", "--kernel", "lt_grad_f64_kernel",
                        "--workload", "s", "--mode", "fp64", "--json", str(js)], input=CSV, capture_output=True, text=True, cwd=ROOT)
    e = json.load(open(js))["captures"]["s/fp64"]
    assert r.returncode == 0 and e["launches_summed"] == 2 and e["dram_bytes_read"] == 104867 and e["dram_bytes_write"] == 268435476
    assert e["duration_ns_under_ncu"] == 68000500


def test_bench_reports_the_step_traffic_of_the_constant_bank_kernels():
    """profiles/ncu_traffic.json as committed: the fp64 headline entry is the sum over the launches of one step and says so."""
    sys.path.insert(0, ROOT)
    import bench
    t = bench.ncu_traffic("cfg3_4096x4096_1000", "fp64")
    assert t is not None and t["launches_summed"] == 3 and "const" in t["kernel"] and "note" in t
    assert t["bytes"] == t["read"] + t["write"] > 3 * 4096 * 4096 * 16 * 0.7      # three writes of the map (+ two re-reads)
    s = bench.ncu_traffic("sie_paper_6730x6730_702", "fp64")
    assert s is not None and "launches_summed" not in s
