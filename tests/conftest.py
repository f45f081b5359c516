import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    """A hung kernel must not hang the suite: every test gets a wall-clock limit (pytest-timeout, if installed)."""
    import pytest
    if not config.pluginmanager.hasplugin("timeout"):
        return
    for item in items:
        if item.get_closest_marker("timeout") is None:
            item.add_marker(pytest.mark.timeout(900))


def pytest_terminal_summary(terminalreporter):
    """O12: print err_normwise and err_elementwise_floored of every GEMV / GEMM case the session checked (worst first per tag
    prefix), and keep the full list where a GPU run can bring it back (gpurun_out/parity_errors.txt)."""
    from util import ERRLOG
    if not ERRLOG:
        return
    tr = terminalreporter
    tr.section("O12 errors of the GEMV / GEMM cases (contract: norm-wise <= 2e-2 bf16, <= 1e-5 fp32)")
    worst = {}
    for tag, dt, en, ee, w in ERRLOG:
        k = (tag.split(":")[0], dt)
        if k not in worst or en > worst[k][0]:
            worst[k] = (en, ee, w, tag)
    for (grp, dt), (en, ee, w, tag) in sorted(worst.items()):
        tr.write_line(f"{grp:28s} {dt:5s} err_normwise {en:.3e}  err_elementwise_floored {ee:.3e}  worst/bound {w:.3f}  ({tag})")
    tr.write_line(f"{len(ERRLOG)} cases checked")
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "parity_errors.txt"), "w") as f:
            f.write("tag dtype err_normwise err_elementwise_floored worst_over_bound\n")
            for tag, dt, en, ee, w in ERRLOG:
                f.write(f"{tag} {dt} {en:.4e} {ee:.4e} {w:.4f}\n")
