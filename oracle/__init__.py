"""ORACLE — test infrastructure only (see mkfo.h). Import allowed from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs; never from the product package."""
