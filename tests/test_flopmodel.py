"""The roofline numerator (host logic): pinned to the per-class table of SURVEY.md section 8d."""
from paper_2406_14920_b200 import flopmodel as fm


def test_flop_model_matches_survey_table():
    # class: (Boys, R build, ERI E-transform, digestion)  -- SURVEY.md section 8d
    table = {(0, 0, 0, 0): (32, 0, 4, 12), (0, 1, 0, 1): (36, 36, 84, 108), (1, 1, 1, 1): (40, 195, 1254, 972),
             (0, 2, 0, 2): (40, 195, 672, 432), (2, 2, 2, 2): (48, 1458, 47712, 15552),
             (0, 3, 3, 3): (50, 2115, 88000, 12000), (2, 3, 2, 3): (52, 2970, 189312, 43200),
             (3, 3, 3, 3): (56, 5421, 706560, 120000)}
    for ls, (b, r, e, d) in table.items():
        f = fm.quartet_flops(*ls)
        assert (f["boys"], f["rbuild"], f["eri"], f["digest"]) == (b, r, e, d), ls


def test_counts_from_the_paper():
    assert len(fm.CLASS_L) == 10                          # 10 pair classes
    assert sum(1 for a in range(10) for b in range(a, 10)) == 55
    assert fm.ncart(1) ** 2 == 9                          # a PP pair = 9 pGTO pairs
    assert fm.ncart(1) * fm.ncart(2) == 18                # a PD pair <-> 18 density elements
    assert fm.ncart(3) ** 2 == 100                        # an FF block = 100 components
    assert [fm.nherm(L) for L in (0, 1, 2, 12)] == [1, 4, 10, 455]
