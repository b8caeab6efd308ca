"""ORACLE — test infrastructure only.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  The product package
(paper_2606_09643_b200) never does, and has no CPU fallback."""
