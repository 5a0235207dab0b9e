"""Host logic of bench.py that needs no device: the nvidia-smi clock samples are filtered to the timed region
(the contract's "clocks" key: median SM clock under load, maximum clock, throttle reasons)."""
import datetime
import importlib.util
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def sampler(bench, t0, t1):
    s = bench.ClockSampler.__new__(bench.ClockSampler)      # no nvidia-smi process: only the parsing is under test
    s.t0, s.t1, s.p = t0, t1, None
    return s


def line(t, sm, reasons=("Not Active",) * 4, active="0x0"):
    return ", ".join([t.strftime("%Y/%m/%d %H:%M:%S.%f")[:-3], str(sm), "1965", "900.0", active, *reasons])


def test_clock_samples_are_filtered_to_the_timed_region():
    bench = load_bench()
    t0 = datetime.datetime(2026, 1, 1, 12, 0, 0)
    dt = datetime.timedelta(milliseconds=100)
    capped = ("Not Active", "Not Active", "Not Active", "Active")
    text = "\n".join([
        line(t0 - 5 * dt, 1200),                             # warm-up: outside
        line(t0 + 1 * dt, 1950, capped),
        line(t0 + 2 * dt, 1965),
        line(t0 + 3 * dt, 1935),
        line(t0 + 9 * dt, 600),                              # after the timed region: outside
        "garbage line",
    ])
    out = sampler(bench, t0, t0 + 4 * dt).summarize(text)
    assert out["samples"] == 3 and out["sm_mhz"] == 1950.0 and out["sm_max_mhz"] == 1965.0
    assert out["reasons"] == ["sw_power_cap"] and out["window"] == "timed region"


def test_a_timed_region_without_a_sample_falls_back_to_the_whole_run_and_says_so():
    bench = load_bench()
    t0 = datetime.datetime(2026, 1, 1, 12, 0, 0)
    text = line(t0 - datetime.timedelta(milliseconds=300), 1965)
    out = sampler(bench, t0, t0 + datetime.timedelta(milliseconds=1)).summarize(text)
    assert out["samples"] == 1 and out["sm_mhz"] == 1965.0 and out["window"].startswith("whole run")
    empty = sampler(bench, t0, t0).summarize("")
    assert empty["samples"] == 0 and empty["sm_mhz"] is None and empty["reasons"] == []
