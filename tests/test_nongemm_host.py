"""Host logic of include/dpi_nongemm.h that needs no GPU: dpi_bfs_schedule (Algorithm 2) must equal
the oracle's step-by-step queue bit for bit."""
import pytest

import oracle
from paper_2606_21101_b200 import build, nongemm


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


@pytest.mark.parametrize("ne", range(0, 9))
def test_bfs_schedule_equals_oracle_queue_on_a_grid(ne):
    for ni in range(0, 9):
        assert nongemm.bfs_schedule(ne, ni) == oracle.bfs_queue(ne, ni), (ne, ni)


def test_bfs_schedule_large_counts():
    for ne, ni in [(1000, 3), (3, 1000), (512, 512), (0, 777)]:
        assert nongemm.bfs_schedule(ne, ni) == oracle.bfs_queue(ne, ni)
