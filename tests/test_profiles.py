"""profiles/traffic.csv (read by bench.py for roofline.traffic) must agree with the ncu summaries it cites: every row names a
summary under profiles/, and the DRAM bytes in that summary (one launch, or the mean over the stage launches it lists) are
the row's.  CPU only."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_traffic_rows_match_the_summaries_they_cite():
    rows = [l.strip() for l in open(os.path.join(ROOT, "profiles", "traffic.csv")) if l.strip()][1:]
    assert rows
    for row in rows:
        workload, variant, nbytes, source = row.split(",", 3)
        path = source.split(" ", 1)[0]
        text = open(os.path.join(ROOT, path)).read()
        per_launch = [float(x) * 1e6 for x in re.findall(r"DRAM bytes per launch \(read \+ write\) \| ([0-9.]+) MB", text)]
        assert per_launch, path
        want = sum(per_launch) / len(per_launch)
        assert abs(float(nbytes) - want) <= 1e-3 * want, (workload, variant, nbytes, want)
        assert workload.split("_")[0] in path


def test_every_profile_names_its_command():
    prof = os.path.join(ROOT, "profiles")
    for name in os.listdir(prof):
        if name.endswith(".md") and name != "traffic.md":
            text = open(os.path.join(prof, name)).read()
            assert "ncu " in text or "bench.py" in text or "cuobjdump" in text, name
        if name.endswith((".csv", ".jsonl", ".json")) and name != "traffic.csv":
            stem = name.rsplit(".", 1)[0]
            assert any(os.path.exists(os.path.join(prof, s + ".md")) for s in (stem, "r02_bench_workloads")), name
