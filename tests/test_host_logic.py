"""Host-side logic of libhec that needs no GPU (-m "not gpu"): the family table of the reduced-polynomial enumeration
(hec_reduced_total) and the partition table of the lambda codes (hec_lambda_partitions), against the oracle."""
import pytest

from oracle import hec_enum_oracle as E
from oracle import hec_lambda_oracle as LO
from paper_1805_11991_b200 import hec


@pytest.mark.parametrize("q,g,d", [(3, 1, 3), (3, 1, 4), (3, 2, 5), (3, 2, 6), (5, 1, 3), (5, 2, 5), (5, 2, 6), (7, 1, 4),
                                   (7, 2, 5), (9, 1, 3), (9, 1, 4), (9, 2, 5), (7, 3, 7), (13, 2, 5)])
def test_reduced_total_equals_the_oracle_enumeration(q, g, d):
    """Same number of reduced polynomials on both sides (they differ only in the choice of coset representatives),
    for p not dividing d and for p | d (reading G19)."""
    assert hec.reduced_total(q, g, d) == sum(1 for _ in E.reduced_polynomials(q, d))


def test_reduced_total_rejects_bad_degrees():
    for q, g, d in [(7, 2, 4), (7, 2, 7), (6, 2, 5), (7, 0, 1)]:
        with pytest.raises(hec.HecError):
            hec.reduced_total(q, g, d)


@pytest.mark.parametrize("g", [1, 2, 3, 4, 5])
def test_lambda_partitions_table(g):
    parts = hec.lambda_partitions(g)
    assert parts == LO.partitions(2 * g + 2)                    # same index order on both sides (hec.h)
    assert all(sum((e + 1) * m for e, m in enumerate(p)) == 2 * g + 2 for p in parts)
    assert len(set(parts)) == len(parts) == [5, 11, 22, 42, 77][g - 1]
