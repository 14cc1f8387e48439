import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device in this container")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


def pytest_sessionfinish(session, exitstatus):
    """GPU runs: keep the worst (max-abs, mean-abs) of every check_attention call per configuration tag."""
    try:
        from parity_util import LIST_REPORT, MAX_ABS_TOL, MEAN_ABS_TOL, REPORT
    except Exception:
        return
    if not REPORT and not LIST_REPORT:
        return
    out = os.path.join(ROOT, "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "gpu_parity_report.txt"), "w") as f:
        f.write(f"# worst attention error per tag over all check_attention calls (budgets: max-abs {MAX_ABS_TOL:g}, mean-abs {MEAN_ABS_TOL:g})\n")
        f.write("tag | checks | worst max-abs | worst mean-abs\n")
        for tag in sorted(REPORT):
            mx, mean, n = REPORT[tag]
            f.write(f"{tag} | {n} | {mx:.3e} | {mean:.3e}\n")
        f.write("# block lists vs oracle: rows, entries, near-ties excused under reading A11 (floored / strict 1e-4 rule); everything else bit-exact\n")
        for tag in sorted(LIST_REPORT):
            st = LIST_REPORT[tag]
            f.write(f"{tag} | rows {st['rows']} | entries {st['entries']} | near-ties floored {st['tie_floored']} | strict {st['tie_strict']}\n")
