"""oracle/ -- TEST INFRASTRUCTURE ONLY (fp64 CPU oracle of the Mesh-Attention compute core).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import anything from here.  Nothing here imports the product package, and the product
package never imports this.
"""
