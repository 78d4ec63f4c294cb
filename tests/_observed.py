"""observed(label, value): print a measured fraction / distance next to the bar that asserts it, tagged with the running test, so
that `pytest -rP` shows how far inside its bar every soft (heuristic-divergence, reading R19) assertion sits and a drift from, say,
99.6 % to 98.1 % identical members is visible although both pass.  The values of the last full run are pinned in DESIGN.md section 8."""
import os


def observed(label, value):
    test = os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0]
    print("\n[observed] %s :: %s = %s" % (test, label, value))
