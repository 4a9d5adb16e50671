"""ORACLE -- test infrastructure only.  A plain, slow NumPy/SciPy CPU
restatement of PAPER.md (arXiv 2202.13532).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import it; the product path
(paper_2202_13532_b200/) never does, and this package never imports the product."""
