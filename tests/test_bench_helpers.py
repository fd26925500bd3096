"""Host-side helpers of bench.py that need no GPU: the digest that ties a stored ncu traffic figure to the kernel sources
it was captured on, and the clock sampler's window logic."""
import importlib
import os
import time


def _bench():
    return importlib.import_module("bench")


def test_traffic_is_only_reported_for_the_sources_it_was_captured_on(tmp_path, monkeypatch):
    bench = _bench()
    digest = bench._csrc_digest()
    assert len(digest) == 16 and int(digest, 16) >= 0 and digest == bench._csrc_digest()
    root = tmp_path
    (root / "profiles").mkdir()
    src = os.path.join(bench.ROOT, "paper_2403_09225_b200")
    os.symlink(src, root / "paper_2403_09225_b200")
    monkeypatch.setattr(bench, "ROOT", str(root))
    # no capture at all
    val, why = bench._stored_traffic(3, "lanes(x)")
    assert val is None and "no ncu capture" in why
    # a capture on other sources: not reported, and the reason says so
    (root / "profiles" / "r01_traffic.csv").write_text("config;kernel_variant;dram_bytes_per_launch\nconfig3;lanes(x);111\n")
    (root / "profiles" / "r02_traffic.csv").write_text(
        "config;kernel_variant;dram_bytes_per_launch;csrc_digest\nconfig3;lanes(x);222;0123456789abcdef\n")
    val, why = bench._stored_traffic(3, "lanes(x)")
    assert val is None and "r02_traffic.csv" in why and "other kernel sources" in why
    # a capture on these sources: reported with its file
    (root / "profiles" / "r03_traffic.csv").write_text(
        f"config;kernel_variant;dram_bytes_per_launch;csrc_digest\nconfig3;lanes(x);333;{digest}\nconfig2;lanes(y);444;{digest}\n")
    val, why = bench._stored_traffic(3, "lanes(x)")
    assert val == 333.0 and "r03_traffic.csv" in why
    assert bench._stored_traffic(2, "lanes(y)")[0] == 444.0
    assert bench._stored_traffic(3, "lanes(other)")[0] is None


def test_clock_sampler_window_picks_the_samples_of_the_region():
    bench = _bench()
    s = bench.ClockSampler(0)
    s.source = "test"
    t0 = time.time()
    s.rows = [(t0 + 0.001 * k, 1965.0 - k, 1965.0, 300.0 + k, ["sw_power_cap"] if k >= 8 else []) for k in range(10)]
    w = s.window(t0 + 0.0025, t0 + 0.0065)        # samples 3, 4, 5, 6
    assert w["samples"] == 4 and w["sm_mhz"] in (1961.0, 1960.0) and w["sm_min_mhz"] == 1959.0 and w["reasons"] == []
    assert w["power_w_max"] == 306.0 and w["sm_max_mhz"] == 1965.0
    w = s.window(t0 + 0.0075, t0 + 0.02)
    assert w["samples"] == 2 and w["reasons"] == ["sw_power_cap"]
    w = s.window(t0 + 0.0041, t0 + 0.0042)          # shorter than the sampling period: nearest samples, flagged
    assert w["samples"] == 2 and "note" in w
    s.source = None
    assert s.window(t0, t0 + 1)["sm_mhz"] is None


def test_digest_ignores_comments_and_white_space_but_not_code():
    import bench
    a = 'int a = 1; // c1\n/* c2\n   c3 */ const char* s = "x // kept /* kept */"; char q = \'"\';  asm("mov // x;");\n\tint   b;'
    assert bench._strip_comments(a) == 'int a = 1; const char* s = "x // kept /* kept */"; char q = \'"\'; asm("mov // x;"); int b;'
    assert bench._strip_comments("x = 1; // one\n") == bench._strip_comments("x  =  1;   /* two */")
    assert bench._strip_comments("x = 1;") != bench._strip_comments("x = 2;")
