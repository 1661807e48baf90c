"""TEST INFRASTRUCTURE: the plain CPU oracle (see pici_oracle.c / pici_oracle.py / ring_oracle.py).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs.  The product package paper_2607_04676_b200 never imports this.
"""
