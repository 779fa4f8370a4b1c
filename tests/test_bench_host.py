"""Host logic of bench.py that needs no GPU: the clock sampler that watches the timed region (one looping nvidia-smi
process, the profiling recipe's form) parses rows, reports throttle reasons and the median clock."""
import importlib.util
import os
import stat
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_under_test", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_clock_sampler_reads_one_looping_process(tmp_path, monkeypatch):
    fake = tmp_path / "nvidia-smi"
    fake.write_text("#!/bin/bash\necho \"$@\" > %s/args\ni=0\nwhile true; do i=$((i+1)); "
                    "if [ $i -le 2 ]; then echo '1200, 1965, Not Active, Not Active, Not Active, Not Active'; "
                    "else echo '1965, 1965, Not Active, Not Active, Not Active, Active'; fi; sleep 0.1; done\n" % tmp_path)
    fake.chmod(fake.stat().st_mode | stat.S_IEXEC)
    monkeypatch.setenv("PATH", str(tmp_path) + os.pathsep + os.environ["PATH"])
    c = _bench().ClockSampler(0)
    c.start()
    time.sleep(1.0)
    c.stop()
    s = c.summary()
    assert "-lms 200" in (tmp_path / "args").read_text()          # one process in loop mode, not one per sample
    assert c.proc.poll() is not None                               # killed after the timed region
    assert s["samples"] >= 5 and s["sm_mhz"] == 1965 and s["sm_max_mhz"] == 1965
    assert s["reasons"] == ["sw_power_cap"]


def test_clock_sampler_without_nvidia_smi(tmp_path, monkeypatch):
    monkeypatch.setenv("PATH", str(tmp_path))                      # no nvidia-smi anywhere: an empty summary, no exception
    c = _bench().ClockSampler(0)
    c.start()
    c.stop()
    assert c.summary() == {"sm_mhz": 0, "sm_max_mhz": 0, "reasons": [], "samples": 0}
