"""CPU oracle of the TPC sector tracker -- TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  The product package (paper_1709_00618_b200) never does.
"""
