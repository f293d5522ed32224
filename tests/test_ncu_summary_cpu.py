"""The ncu raw-page parser (paper_2511_02328_b200/ncu_summary.py) on a small made-up page in ncu's CSV layout
(header row, units row, one row per launch): means per launch, unit scaling, traffic.json entry."""
import json
import subprocess
import sys

RAW = '''"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","dram__bytes_read.sum","dram__bytes_write.sum","gpu__time_duration.sum","launch__registers_per_thread","smsp__thread_inst_executed.sum","smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio"
"","","","","","","","","","","","Gbyte","Mbyte","msecond","register/thread","inst",""
"0","1","python","box","ddsp_interleave_kernel<0>(PreArgs)","1","7","(256, 1, 1)","(10, 1, 1)","0","10.0","1.0","500","2.0","40","1000","0.1"
"1","1","python","box","ddsp_lanes_kernel<0, 1>(LanesArgs)","1","7","(512, 1, 1)","(148, 1, 1)","0","10.0","2.0","1,000","10.0","128","8000","0.5"
"2","1","python","box","ddsp_lanes_kernel<0, 1>(LanesArgs)","1","7","(512, 1, 1)","(148, 1, 1)","0","10.0","4.0","3,000","30.0","128","12000","1.5"
'''


def test_ncu_summary_means_units_and_traffic(tmp_path):
    raw = tmp_path / "raw.csv"
    raw.write_text(RAW)
    md, tr = tmp_path / "s.md", tmp_path / "traffic.json"
    subprocess.check_call([sys.executable, "-m", "paper_2511_02328_b200.ncu_summary", str(raw), "--match", "lanes_kernel",
                           "--kernel", "lanes", "--config", "fast", "--command", "ncu ... made up", "--md", str(md),
                           "--traffic", str(tr), "--adds-per-launch", "20000"])
    t = json.load(open(tr))["lanes/fast"]
    assert t["launches"] == 2
    assert abs(t["dram_bytes_per_launch"] - (3.0e9 + 2000.0e6)) < 1.0        # mean read 3 GB + mean write 2000 MB
    text = md.read_text()
    assert "| duration (`gpu__time_duration.sum`) | 0.02 | msecond |" in text
    assert "long_scoreboard" in text and "instructions per nominal add = 0.5000" in text
