"""Both schedulers against the stored digests of tests/golden/sched_digests.txt (written by
tests/golden/make_golden.py from the reference scheduler alone)."""
import pytest

from paper_2606_09061_b200 import binding, build
from tests.golden import make_golden as mg


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


@pytest.mark.parametrize("name", sorted(mg.CASES))
def test_reference_scheduler_matches_golden(name):
    assert mg.reference_digest(name) == mg.read_golden()[name]


@pytest.mark.parametrize("name", sorted(mg.CASES))
def test_cpp_scheduler_matches_golden(name):
    make_trace, kw = mg.CASES[name]
    cpp = binding.Scheduler(**{**kw, "max_batch": kw.get("S_max", 1024)})
    for rid, a, p, o in zip(*make_trace()):
        cpp.cp_sched_add_request(int(rid), int(a), int(p), int(o))

    def nxt(t):
        cpp.cp_sched_next(t)
        return cpp.batch()

    assert mg.drive(nxt, cpp.cp_sched_commit, cpp.cp_sched_has_work, cpp.cp_sched_next_arrival) == mg.read_golden()[name]
